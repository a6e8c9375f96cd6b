"""GPU parity tests: the CUDA path (through the C-ABI) against the CPU oracle, element by element on
the same seeded inputs.  Bar (BASELINE.json north_star): relative L2 error <= 1e-12 for complex128
and <= 1e-5 for complex64; the stick map is compared for equality in tests/test_host_cabi.py.
"""
import numpy as np
import pytest

from paper_2406_05577_b200 import workloads as wl

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def _rel(a, b):
    a = np.asarray(a, dtype=np.complex128).ravel()
    b = np.asarray(b, dtype=np.complex128).ravel()
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


@pytest.fixture(scope="module")
def fb():
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2406_05577_b200 import binding

    binding.lib()  # fails loudly if libfftb.so is missing
    return binding


def _plan(fb, w, batch, scale="forward", dense=False, host=False):
    p = fb.Plan(w.n, w.cutoff, batch=batch, dtype=w.dtype, scale=scale, dense=dense)
    p.bind(host_staging=host)
    return p


def _small(n, a, dtype="c128", batch=3, dist="uniform", number=0):
    return wl.Workload(number, "t", n, a, dtype, batch, dist, "inv_fwd")


SMALL = [
    _small((32, 32, 32), (8, 8, 8), number=1),
    _small((32, 32, 32), (5, 8, 3)),
    _small((64, 64, 64), (16, 16, 16), batch=5),
    _small((64, 64, 32), (9, 16, 8)),
    _small((32, 32, 96), (8, 8, 24)),
    _small((96, 96, 192), (24, 24, 48), dtype="c64", batch=2, number=4),
    _small((96, 96, 64), (24, 20, 16), dtype="c128", batch=2),
    _small((32, 32, 192), (8, 8, 48), dtype="c128", batch=2),
    _small((128, 128, 128), (32, 32, 32), batch=3, dist="normal_decay", number=3),
    _small((128, 128, 64), (32, 17, 16), dtype="c64", batch=2),
    _small((192, 192, 32), (48, 48, 8), dtype="c64", batch=2),
    _small((192, 192, 32), (48, 40, 8), dtype="c128", batch=1),
    _small((256, 256, 256), (64, 64, 64), batch=1, number=5),
    _small((256, 256, 32), (64, 64, 8), dtype="c64", batch=2),
    _small((256, 256, 64), (40, 50, 16), dtype="c128", batch=2),   # four-way split kernels, partly filled columns
]
IDS = [f"{w.n[0]}x{w.n[1]}x{w.n[2]}-a{w.cutoff[0]}.{w.cutoff[1]}.{w.cutoff[2]}-{w.dtype}" for w in SMALL]


@pytest.mark.parametrize("w", SMALL, ids=IDS)
def test_inverse_forward_vs_oracle(fb, oracle, w):
    p = _plan(fb, w, w.batch)
    k = p.points()
    ko = oracle.enum_points(w.n, w.cutoff)
    assert all(np.array_equal(x, y) for x, y in zip(k, ko))
    c = wl.coefficients(w, *k)
    d_c = torch.from_numpy(c).cuda()
    d_psi = p.inverse(d_c)
    torch.cuda.synchronize()
    psi_ref = oracle.inverse(w.n, ko, c)
    e_inv = _rel(d_psi.cpu().numpy(), psi_ref)
    assert e_inv <= w.tol, f"inverse rel L2 {e_inv:.3e}"
    # the input must be preserved
    assert torch.equal(d_c.cpu(), torch.from_numpy(c))
    # forward of a generic (not band-limited) cuboid
    g = wl.cuboid(w)
    d_g = torch.from_numpy(g).cuda()
    d_f = p.forward(d_g)
    torch.cuda.synchronize()
    C = float(np.prod(w.n))
    f_ref = oracle.forward(w.n, ko, g, 1.0 / C)
    e_fwd = _rel(d_f.cpu().numpy(), f_ref)
    assert e_fwd <= w.tol, f"forward rel L2 {e_fwd:.3e}"
    assert torch.equal(d_g.cpu(), torch.from_numpy(g))
    # round trip recovers the sphere
    d_rt = p.forward(d_psi)
    torch.cuda.synchronize()
    e_rt = _rel(d_rt.cpu().numpy(), c)
    assert e_rt <= w.tol, f"round trip rel L2 {e_rt:.3e}"
    p.destroy()


@pytest.mark.parametrize("w", [SMALL[0], SMALL[2], SMALL[3], SMALL[5], SMALL[8], SMALL[10], SMALL[13], SMALL[14]],
                         ids=[IDS[i] for i in (0, 2, 3, 5, 8, 10, 13, 14)])
def test_apply_vloc_vs_oracle(fb, oracle, w):
    p = _plan(fb, w, w.batch)
    k = p.points()
    c = wl.coefficients(w, *k)
    v = wl.potential(w)
    d_c, d_v = torch.from_numpy(c).cuda(), torch.from_numpy(v).cuda()
    d_o = p.apply_vloc(d_c, d_v)
    torch.cuda.synchronize()
    C = float(np.prod(w.n))
    ref = oracle.apply_vloc(w.n, k, c, v, 1.0 / C)
    e = _rel(d_o.cpu().numpy(), ref)
    assert e <= w.tol, f"vloc rel L2 {e:.3e}"
    # in place (d_packed_in == d_packed_out is allowed)
    d_io = d_c.clone()
    p.apply_vloc(d_io, d_v, d_io)
    torch.cuda.synchronize()
    assert _rel(d_io.cpu().numpy(), ref) <= w.tol
    p.destroy()


DEGENERATE = [((64, 64, 64), (0, 0, 0)), ((64, 64, 64), (1, 1, 1)), ((128, 128, 128), (2, 1, 3)), ((32, 32, 32), (1, 8, 1)),
              ((128, 128, 128), (0, 5, 0)), ((256, 256, 64), (1, 1, 1)), ((256, 256, 256), (0, 0, 7)), ((96, 96, 64), (0, 24, 0)),
              ((128, 128, 128), (32, 0, 0)), ((256, 256, 32), (64, 1, 0))]


@pytest.mark.timeout(120)
@pytest.mark.parametrize("dtype", ["c128", "c64"])
@pytest.mark.parametrize("n,a", DEGENERATE, ids=[f"{n[0]}x{n[1]}x{n[2]}-a{a[0]}.{a[1]}.{a[2]}" for n, a in DEGENERATE])
def test_degenerate_spheres(fb, oracle, n, a, dtype):
    """The degenerate cut-offs: a single point, a single stick, a single column, a single plane of sticks,
    columns that all hold one stick (no y task at all in the persistent kernels)."""
    w = _small(n, a, dtype=dtype, batch=2)
    p = _plan(fb, w, w.batch)
    k = p.points()
    assert all(np.array_equal(x, y) for x, y in zip(k, oracle.enum_points(n, a)))
    c = wl.coefficients(w, *k)
    d_c = torch.from_numpy(c).cuda()
    d_psi = p.inverse(d_c)
    torch.cuda.synchronize()
    assert _rel(d_psi.cpu().numpy(), oracle.inverse(n, k, c)) <= w.tol
    C = float(np.prod(n))
    g = wl.cuboid(w)
    d_f = p.forward(torch.from_numpy(g).cuda())
    v = wl.potential(w)
    d_o = p.apply_vloc(d_c, torch.from_numpy(v).cuda())
    torch.cuda.synchronize()
    assert _rel(d_f.cpu().numpy(), oracle.forward(n, k, g, 1.0 / C)) <= w.tol
    assert _rel(d_o.cpu().numpy(), oracle.apply_vloc(n, k, c, v, 1.0 / C)) <= w.tol
    p.destroy()


def test_scale_none(fb, oracle):
    w = SMALL[0]
    p = _plan(fb, w, w.batch, scale="none")
    k = p.points()
    c = wl.coefficients(w, *k)
    d_rt = p.forward(p.inverse(torch.from_numpy(c).cuda()))
    torch.cuda.synchronize()
    assert _rel(d_rt.cpu().numpy(), float(np.prod(w.n)) * c) <= w.tol  # forward(inverse(c)) = C c (R2)


def test_closed_forms_on_gpu(fb):
    """Impulse -> ones, single plane wave -> exp(+2 pi j k0.i/N) (Eq. 8), without the oracle."""
    w = SMALL[2]
    p = _plan(fb, w, 2)
    k = p.points()
    S = p.S
    c = np.zeros((2, S), np.complex128)
    c[0, (S - 1) // 2] = 1.0
    p0 = 1234
    c[1, p0] = 1.0
    psi = p.inverse(torch.from_numpy(c).cuda()).cpu().numpy()
    assert np.abs(psi[0] - 1).max() < 1e-13
    i3, i2, i1 = np.meshgrid(*[np.arange(w.n[d]) for d in (2, 1, 0)], indexing="ij")
    ref = np.exp(2j * np.pi * (k[0][p0] * i1 / w.n[0] + k[1][p0] * i2 / w.n[1] + k[2][p0] * i3 / w.n[2]))
    assert np.abs(psi[1] - ref).max() < 1e-13


def test_batch_chunking_and_partial_batches(fb, oracle):
    """nb smaller than, equal to and not a multiple of the plan's chunk size; plan reuse."""
    w = _small((64, 64, 64), (16, 16, 16), batch=37)
    p = _plan(fb, w, 37)
    k = p.points()
    c = wl.coefficients(w, *k)
    d_c = torch.from_numpy(c).cuda()
    ref = oracle.inverse(w.n, k, c[:5])
    for nb in (1, 5, 37):
        d_psi = p.inverse(d_c[:nb].contiguous())
        torch.cuda.synchronize()
        m = min(nb, 5)
        assert _rel(d_psi[:m].cpu().numpy(), ref[:m]) <= w.tol
        rt = p.forward(d_psi)
        torch.cuda.synchronize()
        assert _rel(rt.cpu().numpy(), c[:nb]) <= w.tol
    assert p.info["ring_bands"] == 0 and p.last_launches() == 2 * -(-37 // p.info["chunk_bands_fwd"])  # the last call was a forward
    with pytest.raises(fb.FftbError):
        p.inverse(torch.zeros((38, p.S), dtype=torch.complex128, device="cuda"))


def test_host_buffer_calls(fb, oracle):
    w = SMALL[2]
    p = _plan(fb, w, w.batch, host=True)
    k = p.points()
    c = wl.coefficients(w, *k)
    h_c = torch.from_numpy(c).pin_memory()
    d_psi = torch.empty(p.cuboid_shape(w.batch), dtype=torch.complex128, device="cuda")
    p.inverse_host(h_c, d_psi)
    h_rt = torch.empty_like(h_c).pin_memory()
    p.forward_host(d_psi, h_rt)
    torch.cuda.synchronize()
    assert _rel(h_rt.numpy(), c) <= w.tol
    v = wl.potential(w)
    h_o = torch.empty_like(h_c).pin_memory()
    p.apply_vloc_host(h_c, h_o, torch.from_numpy(v).cuda())
    torch.cuda.synchronize()
    ref = oracle.apply_vloc(w.n, k, c, v, 1.0 / float(np.prod(w.n)))
    assert _rel(h_o.numpy(), ref) <= w.tol
    # without the staging area the host calls are refused
    p2 = _plan(fb, w, w.batch, host=False)
    with pytest.raises(fb.FftbError):
        p2.inverse_host(h_c, d_psi)


@pytest.mark.parametrize("dtype", ["c128", "c64"])
@pytest.mark.parametrize("n,a", [((32, 32, 32), (8, 8, 8)), ((64, 64, 64), (16, 16, 16)), ((128, 128, 128), (32, 32, 32)),
                                 ((256, 256, 256), (64, 64, 64))])
def test_pruned_vs_dense(fb, oracle, n, a, dtype):
    """BASELINE config 5: the same data zero-padded to the full cuboid and transformed unpruned by
    the product's kernels gives the same result as the pruned path."""
    w = _small(n, a, dtype=dtype, batch=1 if n[0] >= 128 else 2)
    pp = _plan(fb, w, w.batch)
    pd = _plan(fb, w, w.batch, dense=True)
    k = pp.points()
    c = wl.coefficients(w, *k)
    d_c = torch.from_numpy(c).cuda()
    d_dense_in = pp.dense_embed(pd, d_c)
    psi_p = pp.inverse(d_c)
    psi_d = pd.inverse(d_dense_in)
    torch.cuda.synchronize()
    # embedding is a pure scatter: bit-exact against the oracle-side definition
    cube = np.zeros((w.batch,) + tuple(n), w.complex_dtype)  # [b][k1+N1/2][k2+N2/2][k3+N3/2]
    cube[:, k[0] + n[0] // 2, k[1] + n[1] // 2, k[2] + n[2] // 2] = c
    assert np.array_equal(d_dense_in.cpu().numpy().reshape(cube.shape), cube)
    assert _rel(psi_d.cpu().numpy(), psi_p.cpu().numpy()) <= w.tol
    if n[0] <= 128:
        assert _rel(psi_d.cpu().numpy(), oracle.inverse(n, k, c)) <= w.tol
    back_d = pp.dense_extract(pd, pd.forward(psi_d))
    back_p = pp.forward(psi_p)
    torch.cuda.synchronize()
    assert _rel(back_d.cpu().numpy(), c) <= w.tol and _rel(back_p.cpu().numpy(), c) <= w.tol


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_full_size_configs_sampled_bands(fb, oracle, cfg):
    """BASELINE.json's five configurations at full batch size, in the launch configuration bench.py
    times; the oracle checks a sample of bands (every band is an independent transform)."""
    w = wl.WORKLOADS[cfg]
    p = _plan(fb, w, w.batch)
    k = p.points()
    c = wl.coefficients(w, *k)
    d_c = torch.from_numpy(c).cuda()
    sample = sorted({0, w.batch // 2, w.batch - 1})
    C = float(np.prod(w.n))
    if w.op == "vloc":
        v = wl.potential(w)
        d_o = p.apply_vloc(d_c, torch.from_numpy(v).cuda())
        torch.cuda.synchronize()
        ref = oracle.apply_vloc(w.n, k, c[sample], v, 1.0 / C)
        assert _rel(d_o[sample].cpu().numpy(), ref) <= w.tol
    else:
        d_psi = p.inverse(d_c)
        d_rt = p.forward(d_psi)
        torch.cuda.synchronize()
        ref = oracle.inverse(w.n, k, c[sample])
        assert _rel(d_psi[sample].cpu().numpy(), ref) <= w.tol
        assert _rel(d_rt.cpu().numpy(), c) <= w.tol
        # the persistent kernels hand data between warps through shared memory and mbarriers: repeat the
        # full batch and look at EVERY band, so that a timing-dependent race shows up as one bad band
        for _ in range(3):
            d_psi2 = p.inverse(d_c)
            d_rt2 = p.forward(d_psi2)
            torch.cuda.synchronize()
            assert torch.equal(d_psi2, d_psi)
            err = (d_rt2 - d_c).abs().amax(dim=1) / d_c.abs().amax(dim=1)
            assert float(err.max()) <= 100 * w.tol, f"band {int(err.argmax())}: {float(err.max()):.3e}"
        # Parseval at full size: sum |psi|^2 = C sum |c|^2 (holds at any size)
        e_psi = float((d_psi.abs() ** 2).sum().item())
        e_c = float((np.abs(c.astype(np.complex128)) ** 2).sum())
        assert abs(e_psi - C * e_c) <= 1e-6 * C * e_c


@pytest.mark.parametrize("n,radius,centre,dtype,trim", [((64, 64, 64), 11, (2, -3, 4), "c128", 7), ((128, 128, 128), 27, (-3, 4, 2), "c128", None),
                                                        ((32, 32, 96), 6, (1, 1, -9), "c64", 3), ((96, 96, 64), 13, (3, -2, 1), "c128", 5)])
def test_explicit_stick_map_vs_oracle(fb, oracle, n, radius, centre, dtype, trim):
    """plans from an explicit stick map, here a k-point-shifted
    ball with (optionally) randomly shortened sticks, against the oracle's plain definition evaluated on
    the point list the TEST expands from the map."""
    from test_host_cabi import _shifted_ball_map

    sm = _shifted_ball_map(n, radius, centre, trim_seed=trim)
    nb = 3
    p = fb.Plan(n, batch=nb, dtype=dtype, stick_map=sm).bind()
    rep = np.repeat(np.arange(sm[0].size), sm[3])
    off = np.concatenate([[0], np.cumsum(sm[3])])[:-1]
    k = (sm[0][rep], sm[1][rep], (sm[2][rep] + (np.arange(rep.size) - off[rep])).astype(np.int32))
    assert all(np.array_equal(a, b) for a, b in zip(p.points(), k))
    w = wl.Workload(0, "explicit", n, (0, 0, 0), dtype, nb, "uniform", "inv_fwd")
    c = wl.coefficients(w, *k)
    d_c = torch.from_numpy(c).cuda()
    d_psi = p.inverse(d_c)
    torch.cuda.synchronize()
    assert _rel(d_psi.cpu().numpy(), oracle.inverse(n, k, c)) <= w.tol
    g = wl.cuboid(w)
    d_f = p.forward(torch.from_numpy(g).cuda())
    torch.cuda.synchronize()
    C = float(np.prod(n))
    assert _rel(d_f.cpu().numpy(), oracle.forward(n, k, g, 1.0 / C)) <= w.tol
    v = wl.potential(w)
    d_o = p.apply_vloc(d_c, torch.from_numpy(v).cuda())
    torch.cuda.synchronize()
    assert _rel(d_o.cpu().numpy(), oracle.apply_vloc(n, k, c, v, 1.0 / C)) <= w.tol
    p.destroy()


def test_explicit_map_many_single_stick_columns_256(fb, oracle):
    """An explicit map on a 256 x 256 grid whose k1 columns mostly hold ONE stick (more such columns than
    the plane kernels have warps): they take the closed-form path of the four-way-split kernels."""
    n = (256, 256, 32)
    k1, k2, k3lo, ln = [], [], [], []
    for a in range(-21, 22):
        run = range(-4, 5) if abs(a) <= 3 else [a % 7 - 3]
        for b in run:
            k1.append(a); k2.append(b); k3lo.append(-3 - (a + b) % 3); ln.append(5 + (a * b) % 4)
    sm = tuple(np.asarray(x, dtype=np.int32) for x in (k1, k2, k3lo, ln))
    nb = 2
    p = fb.Plan(n, batch=nb, dtype="c128", stick_map=sm).bind()
    k = p.points()
    w = wl.Workload(0, "explicit", n, (0, 0, 0), "c128", nb, "uniform", "inv_fwd")
    c = wl.coefficients(w, *k)
    d_c = torch.from_numpy(c).cuda()
    d_psi = p.inverse(d_c)
    torch.cuda.synchronize()
    assert _rel(d_psi.cpu().numpy(), oracle.inverse(n, k, c)) <= w.tol
    C = float(np.prod(n))
    g = wl.cuboid(w)
    d_f = p.forward(torch.from_numpy(g).cuda())
    v = wl.potential(w)
    d_o = p.apply_vloc(d_c, torch.from_numpy(v).cuda())
    torch.cuda.synchronize()
    assert _rel(d_f.cpu().numpy(), oracle.forward(n, k, g, 1.0 / C)) <= w.tol
    assert _rel(d_o.cpu().numpy(), oracle.apply_vloc(n, k, c, v, 1.0 / C)) <= w.tol
    p.destroy()


def _explicit_256_case(fb, oracle, sm, n, dtype, nb):
    p = fb.Plan(n, batch=nb, dtype=dtype, stick_map=sm).bind()
    k = p.points()
    w = wl.Workload(0, "explicit", n, (0, 0, 0), dtype, nb, "uniform", "inv_fwd")
    c = wl.coefficients(w, *k)
    d_c = torch.from_numpy(c).cuda()
    d_psi = p.inverse(d_c)
    torch.cuda.synchronize()
    assert _rel(d_psi.cpu().numpy(), oracle.inverse(n, k, c)) <= w.tol
    C = float(np.prod(n))
    g = wl.cuboid(w)
    d_f = p.forward(torch.from_numpy(g).cuda())
    v = wl.potential(w)
    d_o = p.apply_vloc(d_c, torch.from_numpy(v).cuda())
    torch.cuda.synchronize()
    assert _rel(d_f.cpu().numpy(), oracle.forward(n, k, g, 1.0 / C)) <= w.tol
    assert _rel(d_o.cpu().numpy(), oracle.apply_vloc(n, k, c, v, 1.0 / C)) <= w.tol
    p.destroy()


@pytest.mark.parametrize("dtype", ["c128", "c64"])
def test_explicit_map_129_multi_stick_columns_256(fb, oracle, dtype):
    """All 129 k1 columns of a 256 x 256 grid hold several sticks: 33 y tasks, one more than the warps' columns of tensor
    memory hold in complex128 -- the plane kernels of the 256 pattern then take their variants without tensor memory
    (running sums of the forward y passes through L2, inputs of the inverse y passes through the landing zone)."""
    n = (256, 256, 32)
    k1, k2, k3lo, ln = [], [], [], []
    for a in range(-64, 65):
        half = 1 + (a % 3) if abs(a) < 60 else 64 - abs(a) + 1  # 3, 5 or 7 sticks; the edge columns up to 11
        for b in range(-half, half + 1):
            k1.append(a); k2.append(b); k3lo.append(-2 - (a + b) % 3); ln.append(4 + (a * b) % 3)
    sm = tuple(np.asarray(x, dtype=np.int32) for x in (k1, k2, k3lo, ln))
    _explicit_256_case(fb, oracle, sm, n, dtype, 2)


def test_explicit_map_singles_between_multi_stick_columns_256(fb, oracle):
    """Single-stick columns BETWEEN multi-stick columns of a 256 x 256 grid, and a column reaching |k2| = 64: the stick
    runs of a y task's four columns are then one contiguous range of the row of A only together with the single sticks
    that lie in between (the inverse plane kernel's one bulk copy per task covers them), and the +N/4 alias of the y axis
    travels through L2 next to the sums in tensor memory."""
    n = (256, 256, 32)
    k1, k2, k3lo, ln = [], [], [], []
    for a in range(-40, 41):
        if a % 3 == 1:
            run = [a % 5 - 2]
        elif a == 0:
            run = range(-64, 65)
        else:
            run = range(-(abs(a) % 29) - 1, (abs(a) % 31) + 2)
        for b in run:
            k1.append(a); k2.append(b); k3lo.append(-3 + (a - b) % 2); ln.append(3 + (a * a + b) % 4)
    sm = tuple(np.asarray(x, dtype=np.int32) for x in (k1, k2, k3lo, ln))
    _explicit_256_case(fb, oracle, sm, n, "c128", 3)


@pytest.mark.parametrize("dtype,nb", [("c128", 37), ("c64", 64), ("c128", 1)])
def test_batch_fastest_packed_layout(fb, oracle, dtype, nb):
    """PAPER.md:219-221 (Fig. 8, "b x y z"): coefficients held with the band index fastest go through
    fftb_packed_transpose: bit-exact transposition both ways (ragged tiles), and the fused local potential
    applied to batch-fastest data equals the oracle's result transposed."""
    w = _small((64, 64, 32), (16, 11, 8), dtype=dtype, batch=nb)
    p = _plan(fb, w, nb)
    k = p.points()
    c = wl.coefficients(w, *k)                                   # [nb][S]
    c_sb = np.ascontiguousarray(c.T)                             # [S][nb], batch fastest
    d_sb = torch.from_numpy(c_sb).cuda()
    d_bs = p.packed_to_band_slowest(d_sb)
    torch.cuda.synchronize()
    assert torch.equal(d_bs.cpu(), torch.from_numpy(c))
    assert torch.equal(p.packed_to_band_fastest(d_bs).cpu(), torch.from_numpy(c_sb))
    v = wl.potential(w)
    d_o = p.packed_to_band_fastest(p.apply_vloc(d_bs, torch.from_numpy(v).cuda()))
    torch.cuda.synchronize()
    ref = oracle.apply_vloc(w.n, k, c, v, 1.0 / float(np.prod(w.n)))
    assert _rel(d_o.cpu().numpy(), np.ascontiguousarray(ref.T)) <= w.tol
    # in place is refused
    with pytest.raises(fb.FftbError):
        p.packed_to_band_slowest(d_sb, out=d_sb.view(nb, p.S))
    p.destroy()


def test_device_calls_are_graph_capturable(fb):
    """fftb_inverse / fftb_forward / fftb_apply_vloc only enqueue kernels on the caller's stream (no allocation,
    no synchronisation), so a caller may capture them in a CUDA graph: replay gives the same bits."""
    w = SMALL[2]
    p = _plan(fb, w, w.batch)
    k = p.points()
    d_c = torch.from_numpy(wl.coefficients(w, *k)).cuda()
    d_v = torch.from_numpy(wl.potential(w)).cuda()
    d_psi = torch.empty(p.cuboid_shape(w.batch), dtype=p.torch_complex, device="cuda")
    d_rt, d_o = torch.empty_like(d_c), torch.empty_like(d_c)

    def step():
        p.inverse(d_c, d_psi)
        p.forward(d_psi, d_rt)
        p.apply_vloc(d_c, d_v, d_o)

    step()
    torch.cuda.synchronize()
    ref = (d_psi.clone(), d_rt.clone(), d_o.clone())
    s = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        step()
        s.synchronize()
        with torch.cuda.graph(g, stream=s):
            step()
    torch.cuda.synchronize()
    for t in (d_psi, d_rt, d_o):
        t.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert all(torch.equal(a, b) for a, b in zip((d_psi, d_rt, d_o), ref))
    del g
    p.destroy()


@pytest.mark.parametrize("dtype", ["c128", "c64"])
def test_host_buffer_calls_pipelined(fb, oracle, dtype):
    """Batches of 32 bands and more cross PCIe in chunks on the plan's copy streams, overlapped with the
    transforms: same results as the device-pointer calls, complete when the caller's stream is.  complex64: S is
    odd, so the chunks must start on even bands to keep the packed pointers 16-byte aligned (43 * k / 4 is odd)."""
    w = _small((64, 64, 64), (16, 16, 16), batch=43, dtype=dtype)
    p = _plan(fb, w, w.batch, host=True)
    k = p.points()
    c = wl.coefficients(w, *k)
    h_c = torch.from_numpy(c).pin_memory()
    d_psi = torch.empty(p.cuboid_shape(w.batch), dtype=p.torch_complex, device="cuda")
    h_rt = torch.zeros_like(h_c).pin_memory()
    h_o = torch.zeros_like(h_c).pin_memory()
    v = wl.potential(w)
    d_v = torch.from_numpy(v).cuda()
    for _ in range(2):  # twice: the second call must wait for the first one's use of the staging area
        p.inverse_host(h_c, d_psi)
        p.forward_host(d_psi, h_rt)
        p.apply_vloc_host(h_c, h_o, d_v)
    torch.cuda.current_stream().synchronize()
    assert _rel(h_rt.numpy(), c) <= w.tol
    assert torch.equal(d_psi, p.inverse(torch.from_numpy(c).cuda()))
    sample = [0, 21, 42]
    ref = oracle.apply_vloc(w.n, k, c[sample], v, 1.0 / float(np.prod(w.n)))
    assert _rel(h_o.numpy()[sample], ref) <= w.tol


@pytest.mark.parametrize("n,a", [((64, 64, 64), (16, 16, 16)), ((128, 128, 128), (32, 32, 32)), ((96, 96, 192), (24, 24, 48)),
                                 ((64, 64, 256), (16, 16, 64))],
                         ids=["64", "128", "96x96x192", "64x64x256"])
def test_complex64_odd_packed_ranges(fb, oracle, n, a):
    """complex64 z passes move the packed ranges of a tile by 16-byte bulk copies although a range may begin and end on
    an odd 8-byte element: S and nb odd, so ranges of both parities occur and the batch itself ends on an odd element;
    the packed output sits between sentinels that must survive (no store outside [0, nb S))."""
    w = _small(n, a, dtype="c64", batch=3)
    p = _plan(fb, w, 3)
    assert p.S % 2 == 1
    k = p.points()
    c = wl.coefficients(w, *k)
    d_psi = p.inverse(torch.from_numpy(c).cuda())
    torch.cuda.synchronize()
    assert _rel(d_psi.cpu().numpy(), oracle.inverse(w.n, k, c)) <= w.tol
    guard = 2  # complex64 elements = 16 bytes: the view stays 16-byte aligned
    buf = torch.full((guard + 3 * p.S + guard,), 777.0 - 555.0j, dtype=torch.complex64, device="cuda")
    out = buf[guard:guard + 3 * p.S].view(3, p.S)
    p.forward(d_psi, out)
    torch.cuda.synchronize()
    h = buf.cpu().numpy()
    assert (h[:guard] == np.complex64(777.0 - 555.0j)).all() and (h[-guard:] == np.complex64(777.0 - 555.0j)).all()
    assert _rel(h[guard:-guard].reshape(3, p.S), c) <= w.tol
    p.destroy()


def test_complex64_odd_band_chunks(fb, oracle):
    """A workspace budget of one band (fftb_plan_tuning.workspace_bytes) makes the library run band by band: with
    complex64 and an odd S every second chunk's packed pointer is only 8-byte aligned, which the bulk copies of the z
    passes must cope with."""
    w = _small((128, 128, 128), (32, 32, 32), dtype="c64", batch=3)
    p = fb.Plan(w.n, w.cutoff, batch=3, dtype="c64", tuning={"workspace_bytes": 4 << 20}).bind()
    assert p.info["chunk_bands"] == 1 and p.S % 2 == 1 and p.info["ring_bands"] == 0
    k = p.points()
    c = wl.coefficients(w, *k)
    d_psi = p.inverse(torch.from_numpy(c).cuda())
    rt = p.forward(d_psi)
    torch.cuda.synchronize()
    assert p.last_launches() == 6
    assert _rel(d_psi.cpu().numpy(), oracle.inverse(w.n, k, c)) <= w.tol
    assert _rel(rt.cpu().numpy(), c) <= w.tol
    p.destroy()
