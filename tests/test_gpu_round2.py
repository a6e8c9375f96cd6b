"""GPU tests added in round 2: the fused launches (z tiles + planes in one cooperative kernel, the intermediate in an
L2-resident ring), stage-level parity through the bind block, the tuning descriptor, band sharding on the CUDA path,
two host threads driving two plans, and the alignment contract.  All comparisons with the oracle use north_star's
bar (relative L2 1e-12 / 1e-5) unless a docstring derives another one."""
import threading

import numpy as np
import pytest

from paper_2406_05577_b200 import workloads as wl
from paper_2406_05577_b200.sharding import band_range

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

    binding.lib()
    return binding


def _w(n, a, dtype="c128", batch=3, dist="uniform", number=0):
    return wl.Workload(number, "t", n, a, dtype, batch, dist, "inv_fwd")


def _intermediate(p, bands):
    """The intermediate A[b][z][stick] of the listed bands (an int = the first so many), read out of the caller-owned
    bind block through the layout fftb_plan_info describes: A[band][z][pitch] for separate launches, tile-major ring
    slots (band b in slot b % ring_bands) for the fused launches."""
    bands = list(range(bands)) if isinstance(bands, int) else list(bands)
    n3, pitch, ns = p.n[2], p.info["pitch"], p.info["n_sticks"]
    elem = 16 if p.dtype == "c128" else 8
    off = p.info["workspace_offset"]
    out = []
    if p.info["ring_bands"] == 0:
        for b in bands:
            raw = p.mem[off + b * n3 * pitch * elem:off + (b + 1) * n3 * pitch * elem]
            out.append(raw.view(p.torch_complex).view(n3, pitch)[:, :ns].cpu().numpy())
        return np.stack(out)
    ts, te, rp, ring = p.info["ring_tile_sticks"], p.info["ring_tile_elems"], p.info["ring_pair_pitch"], p.info["ring_bands"]
    slot = -(-ns // ts) * te
    s, z = np.arange(ns)[None, :], np.arange(n3)[:, None]
    idx = (s // ts) * te + (z // 2) * rp + (z % 2) * ts + s % ts
    for b in bands:
        sl = b % ring
        raw = p.mem[off + sl * slot * elem:off + (sl + 1) * slot * elem].view(p.torch_complex).cpu().numpy()
        out.append(raw[idx])
    return np.stack(out)


# ---------------------------------------------------------------------------------------------------------------
# fused launches
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.timeout(300)
@pytest.mark.parametrize("dtype", ["c128", "c64"])
@pytest.mark.parametrize("nb,ring,lead,zc", [(1, 0, 0, 0), (3, 0, 0, 0), (7, 2, 1, 0), (13, 3, 2, 0), (40, 0, 0, 0), (9, 1, 0, 0),
                                             (1, 0, 0, 20), (13, 3, 2, 24), (40, 0, 0, 16), (9, 1, 0, 40), (6, 2, 1, 147), (6, 2, 1, 1000)])
def test_fused_launch_equals_separate_launches(fb, oracle, dtype, nb, ring, lead, zc):
    """fftb_inverse / fftb_forward as ONE cooperative launch (ring of band slots, per-band counters) do the same
    arithmetic in the same order as the separate z-pass and plane launches: the outputs are bit-identical, for batches
    smaller than, equal to and several times the ring, and for the smallest legal rings (slot reuse on every band).
    zc > 0: the spatial split (zc CTAs walk the z tiles only, the others the planes only; one plane CTA left at 147, and
    a value beyond the grid falls back to the merged walk)."""
    w = _w((128, 128, 128), (32, 32, 32), dtype=dtype, batch=nb, dist="normal_decay", number=3)
    pf = fb.Plan(w.n, w.cutoff, batch=nb, dtype=dtype,
                 tuning={"flags": fb.FFTB_TUNE_FUSED, "ring_bands": ring, "lead_bands": lead, "z_ctas": zc}).bind()
    pu = fb.Plan(w.n, w.cutoff, batch=nb, dtype=dtype).bind()
    assert pf.info["ring_bands"] >= 1 and pu.info["ring_bands"] == 0
    if ring:
        assert pf.info["ring_bands"] == min(ring, nb) and pf.info["lead_bands"] <= max(pf.info["ring_bands"] - 1, 0)
    k = pf.points()
    c = wl.coefficients(w, *k)
    d_c = torch.from_numpy(c).cuda()
    psi_f, psi_u = pf.inverse(d_c), pu.inverse(d_c)
    assert pf.last_launches() == 1 and pu.last_launches() == 2
    torch.cuda.synchronize()
    assert torch.equal(psi_f, psi_u)
    g = torch.from_numpy(wl.cuboid(w, batch=min(nb, 3))).cuda()
    g = g.repeat((nb + g.shape[0] - 1) // g.shape[0], 1, 1, 1)[:nb].contiguous()
    g[nb - 1] *= 0.5  # the last band differs from its copies
    f_f, f_u = pf.forward(g), pu.forward(g)
    torch.cuda.synchronize()
    assert torch.equal(f_f, f_u)
    rt = pf.forward(psi_f)
    torch.cuda.synchronize()
    assert _rel(rt.cpu().numpy(), c) <= w.tol
    sample = sorted({0, nb // 2, nb - 1})
    assert _rel(psi_f[sample].cpu().numpy(), oracle.inverse(w.n, k, c[sample])) <= w.tol
    pf.destroy(); pu.destroy()


@pytest.mark.timeout(300)
def test_fused_launch_repeatable(fb):
    """The counters that order the items are cleared by every call: 20 back-to-back inverse + forward calls on one
    plan, every result bit-identical to the first (a lost wake-up or a slot overwritten too early would show)."""
    w = _w((128, 128, 128), (32, 32, 32), batch=24, dist="normal_decay", number=3)
    p = fb.Plan(w.n, w.cutoff, batch=24, tuning={"flags": fb.FFTB_TUNE_FUSED, "ring_bands": 3, "lead_bands": 2}).bind()
    assert p.info["ring_bands"] == 3
    d_c = torch.from_numpy(wl.coefficients(w, *p.points())).cuda()
    psi0 = p.inverse(d_c).clone()
    rt0 = p.forward(psi0).clone()
    for _ in range(20):
        psi = p.inverse(d_c)
        rt = p.forward(psi)
        torch.cuda.synchronize()
        assert torch.equal(psi, psi0) and torch.equal(rt, rt0)
    p.destroy()


@pytest.mark.parametrize("dtype,nb", [("c128", 43), ("c64", 43), ("c128", 5)])
def test_host_calls_with_deferred_completion(fb, oracle, dtype, nb):
    """FFTB_TUNE_HOST_DEFER: the *_host calls do not make the stream wait for their device-to-host copies and take two
    incoming / two outgoing staging areas in turn; fftb_host_flush closes them all.  Five calls in a row with DIFFERENT
    inputs and outputs (more calls than staging areas: an area rewritten before its copies were done would show), then one
    flush: every output equals what the same plan computes from device pointers, bit for bit, and the oracle within
    tolerance.  43 bands cross PCIe in chunks, 5 bands in one piece."""
    w = _w((64, 64, 64), (16, 16, 16), dtype=dtype, batch=nb, number=2)
    p = fb.Plan(w.n, w.cutoff, batch=nb, dtype=dtype, tuning={"flags": fb.FFTB_TUNE_HOST_DEFER}).bind(host_staging=True)
    plain = fb.Plan(w.n, w.cutoff, batch=nb, dtype=dtype)
    assert p.info["device_bytes_host"] - p.info["device_bytes"] >= 2 * (plain.info["device_bytes_host"] - plain.info["device_bytes"]) - 4096
    plain.destroy()
    k = p.points()
    base = wl.coefficients(w, *k)
    v = wl.potential(w)
    d_v = torch.from_numpy(v).cuda()
    ins = [torch.from_numpy(np.ascontiguousarray(base * (1.0 + 0.25 * i))).pin_memory() for i in range(5)]
    rts = [torch.zeros_like(ins[0]).pin_memory() for _ in range(5)]
    outs = [torch.zeros_like(ins[0]).pin_memory() for _ in range(5)]
    psis = [torch.empty(p.cuboid_shape(nb), dtype=p.torch_complex, device="cuda") for _ in range(5)]
    for i in range(5):
        p.inverse_host(ins[i], psis[i])
        p.forward_host(psis[i], rts[i])
        p.apply_vloc_host(ins[i], outs[i], d_v)
    p.host_flush()
    torch.cuda.current_stream().synchronize()
    for i in range(5):
        d_c = ins[i].cuda()
        assert torch.equal(psis[i], p.inverse(d_c))
        assert torch.equal(rts[i].cuda(), p.forward(psis[i]))
        assert torch.equal(outs[i].cuda(), p.apply_vloc(d_c, d_v))
        assert _rel(rts[i].numpy(), ins[i].numpy()) <= w.tol
    ref = oracle.apply_vloc(w.n, k, ins[3].numpy()[[0, nb - 1]], v, 1.0 / float(np.prod(w.n)))
    assert _rel(outs[3].numpy()[[0, nb - 1]], ref) <= w.tol
    p.host_flush()  # a second flush with nothing new is harmless
    torch.cuda.synchronize()
    p.destroy()


@pytest.mark.timeout(300)
@pytest.mark.parametrize("n,a,dtype,nb", [((256, 256, 128), (64, 64, 32), "c128", 5), ((256, 256, 64), (40, 50, 16), "c64", 6)])
def test_256_pattern_repeatable(fb, n, a, dtype, nb):
    """The plane kernels of the 256 pattern park per-thread values in tensor memory, reuse one shared-memory zone as TMA landing
    zone and staging area and move the cuboid by tensor copies: 12 back-to-back inverse + forward + fused apply calls on one
    plan, every result bit-identical to the first (a zone refilled or a column of tensor memory rewritten too early would
    show), and the round trip recovers the input."""
    w = _w(n, a, batch=nb, dtype=dtype, number=5)
    p = fb.Plan(w.n, w.cutoff, batch=nb, dtype=dtype).bind()
    d_c = torch.from_numpy(wl.coefficients(w, *p.points())).cuda()
    d_v = torch.from_numpy(wl.potential(w)).cuda()
    psi0 = p.inverse(d_c).clone()
    rt0 = p.forward(psi0).clone()
    h0 = p.apply_vloc(d_c, d_v).clone()
    torch.cuda.synchronize()
    assert float((rt0 - d_c).abs().max() / d_c.abs().max()) <= (1e-12 if dtype == "c128" else 1e-5)
    for _ in range(12):
        psi = p.inverse(d_c)
        rt = p.forward(psi)
        h = p.apply_vloc(d_c, d_v)
        torch.cuda.synchronize()
        assert torch.equal(psi, psi0) and torch.equal(rt, rt0) and torch.equal(h, h0)
    p.destroy()


# ---------------------------------------------------------------------------------------------------------------
# stage-level parity: the intermediate A read back through fftb_plan_info.workspace_offset / pitch
# ---------------------------------------------------------------------------------------------------------------
STAGE = [((64, 64, 64), (16, 16, 16), "c128", {}), ((128, 128, 128), (32, 32, 32), "c128", {}),
         ((128, 128, 128), (32, 32, 32), "c128", {"flags": 4}), ((128, 128, 128), (32, 32, 32), "c64", {"flags": 4}),
         ((256, 256, 256), (64, 64, 64), "c128", {}),
         ((96, 96, 192), (24, 24, 48), "c64", {}), ((32, 32, 32), (8, 8, 8), "c128", {})]


@pytest.mark.parametrize("n,a,dtype,tuning", STAGE, ids=[f"{n[0]}x{n[2]}-{d}-{'fused' if t else 'default'}" for n, a, d, t in STAGE])
def test_stage_parity_inverse_z_and_forward_xy(fb, oracle, n, a, dtype, tuning):
    """After fftb_inverse the bind block holds A[b][z][stick] = the z-only stage of the oracle (its n_axes = 1 output)
    at the stick's (k1 mod N1, k2 mod N2) column: every stick is an independent 1D transform, so the error is measured
    PER STICK relative to that stick's own norm (a misplaced or mis-scaled stick cannot hide behind the others).
    After fftb_forward it holds the x+y stage: for every z-plane the 2D transform of the plane at the stick columns,
    which the oracle computes as its forward on an (N1, N2, 1) grid with the planes as batch."""
    nb = 2
    w = _w(n, a, dtype=dtype, batch=nb)
    p = fb.Plan(n, a, batch=nb, dtype=dtype, scale="none", tuning=tuning or None).bind()
    m = p.get_map()
    k = p.points()
    ns = p.info["n_sticks"]
    c = wl.coefficients(w, *k)
    p.inverse(torch.from_numpy(c).cuda())
    torch.cuda.synchronize()
    A = _intermediate(p, nb).astype(np.complex128)                                   # [b][z][s]
    stage = oracle.inverse(n, k, c, n_axes=1)                                        # [b][i3][i2][i1], z transformed only
    ref = stage[:, :, m["k2"] % n[1], m["k1"] % n[0]]                                # [b][z][s]
    err = np.linalg.norm(A - ref, axis=1) / np.linalg.norm(ref, axis=1)               # per band and stick
    assert err.max() <= w.tol, f"inverse z stage: stick {np.unravel_index(err.argmax(), err.shape)} rel {err.max():.3e}"
    # forward: x+y stage
    g = wl.cuboid(w, batch=nb)
    p.forward(torch.from_numpy(g).cuda())
    torch.cuda.synchronize()
    assert p.info["y_residues"] == 1 or n[0] in (32, 192)
    if p.info["y_residues"] == 1:
        A = _intermediate(p, nb).astype(np.complex128)
        k2d = (m["k1"], m["k2"], np.zeros(ns, np.int32))
        ref = oracle.forward((n[0], n[1], 1), k2d, g.reshape(nb * n[2], 1, n[1], n[0]), 1.0).reshape(nb, n[2], ns)
        assert _rel(A, ref) <= w.tol
    p.destroy()


@pytest.mark.timeout(600)
@pytest.mark.parametrize("fused", [False, True], ids=["default", "fused"])
def test_full_size_config3_stage_per_stick_and_generic_forward(fb, oracle, fused):
    """Config 3 at full batch, in the launch configuration bench.py times (and in the opt-in fused one).  Its
    1/(1+|k|^2) decay makes the whole-output L2 error blind to the high-|k| sticks, so (i) the intermediate of sampled
    bands after the full-batch inverse is compared with the oracle's z-only stage STICK BY STICK; (ii) a full batch of
    generic (not band-limited, seeded on the device) cuboids is transformed forward and two sampled bands are compared
    with the oracle."""
    w = wl.WORKLOADS[3]
    p = fb.Plan(w.n, w.cutoff, batch=w.batch, dtype=w.dtype, tuning={"flags": fb.FFTB_TUNE_FUSED} if fused else None).bind()
    ring = p.info["ring_bands"]
    assert (ring >= 2) == fused
    m, k = p.get_map(), p.points()
    c = wl.coefficients(w, *k)
    d_psi = p.inverse(torch.from_numpy(c).cuda())
    torch.cuda.synchronize()
    sample = [w.batch - 1, w.batch - ring] if fused else [0, 77, w.batch - 1]  # fused: the bands still in the ring
    A = _intermediate(p, sample)
    for got, b in zip(A, sample):
        ref = oracle.inverse(w.n, k, c[b:b + 1], n_axes=1)[0][:, m["k2"] % w.n[1], m["k1"] % w.n[0]]
        err = np.linalg.norm(got - ref, axis=0) / np.linalg.norm(ref, axis=0)
        assert err.max() <= w.tol, f"band {b} stick {err.argmax()}: {err.max():.3e}"
    del d_psi
    gen = torch.Generator(device="cuda").manual_seed(3003)
    g = torch.empty(p.cuboid_shape(w.batch), dtype=torch.complex128, device="cuda")
    torch.view_as_real(g).uniform_(-1.0, 1.0, generator=gen)
    f = p.forward(g)
    torch.cuda.synchronize()
    C = float(np.prod(w.n))
    for b in (5, w.batch - 2):
        ref = oracle.forward(w.n, k, g[b:b + 1].cpu().numpy(), 1.0 / C)
        assert _rel(f[b:b + 1].cpu().numpy(), ref) <= w.tol
    p.destroy()


# ---------------------------------------------------------------------------------------------------------------
# tuning descriptor (replaces the environment variables of round 1)
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,a,dtype", [((64, 64, 64), (16, 16, 16), "c128"), ((128, 128, 128), (32, 32, 32), "c128"),
                                       ((128, 128, 64), (32, 20, 16), "c64"), ((96, 96, 96), (24, 24, 24), "c64")])
@pytest.mark.parametrize("flags", [1, 2, 3], ids=["generic_z", "generic_plane", "generic_both"])
def test_generic_kernels_through_tuning_flags(fb, oracle, n, a, dtype, flags):
    """FFTB_TUNE_GENERIC_Z / _PLANE route a plan through the generic kernels of fftb_kernels.cuh at sizes where a
    persistent kernel exists: all four combinations of z pass and plane kernel agree with the oracle."""
    w = _w(n, a, dtype=dtype, batch=3)
    p = fb.Plan(n, a, batch=3, dtype=dtype, tuning={"flags": flags}).bind()
    k = p.points()
    c = wl.coefficients(w, *k)
    d_c = torch.from_numpy(c).cuda()
    d_psi = p.inverse(d_c)
    torch.cuda.synchronize()
    assert _rel(d_psi.cpu().numpy(), oracle.inverse(n, k, c)) <= w.tol
    g = wl.cuboid(w)
    C = float(np.prod(n))
    d_f = p.forward(torch.from_numpy(g).cuda())
    v = wl.potential(w)
    d_o = p.apply_vloc(d_c, torch.from_numpy(v).cuda())
    torch.cuda.synchronize()
    assert _rel(d_f.cpu().numpy(), oracle.forward(n, k, g, 1.0 / C)) <= w.tol
    assert _rel(d_o.cpu().numpy(), oracle.apply_vloc(n, k, c, v, 1.0 / C)) <= w.tol
    p.destroy()


def test_tuning_is_validated(fb):
    with pytest.raises(fb.FftbError) as e:
        fb.Plan((64, 64, 64), (16, 16, 16), tuning={"flags": 32})  # an unknown flag
    assert e.value.code == fb.FFTB_EINVAL
    with pytest.raises(fb.FftbError) as e:
        fb.Plan((64, 64, 64), (16, 16, 16), tuning={"ring_bands": -1})
    assert e.value.code == fb.FFTB_EINVAL
    with pytest.raises(fb.FftbError) as e:
        fb.Plan((64, 64, 64), (16, 16, 16), tuning={"z_ctas": 1025})
    assert e.value.code == fb.FFTB_EINVAL


# ---------------------------------------------------------------------------------------------------------------
# alignment contract
# ---------------------------------------------------------------------------------------------------------------
def test_misaligned_pointers_are_refused(fb):
    """complex128 cuboids are moved as 32-byte (x, x+1) pairs: a cuboid pointer at 16 mod 32 must come back as
    FFTB_EINVAL instead of raising a misaligned-address fault in the kernel; packed pointers need 16 bytes."""
    import ctypes

    w = _w((64, 64, 64), (16, 16, 16), batch=1)
    p = fb.Plan(w.n, w.cutoff, batch=1).bind()
    L = fb.lib()
    d_c = torch.zeros(p.S + 2, dtype=torch.complex128, device="cuda")
    buf = torch.zeros(int(np.prod(w.n)) + 2, dtype=torch.complex128, device="cuda")
    assert buf.data_ptr() % 32 == 0 and d_c.data_ptr() % 16 == 0
    vp = ctypes.c_void_p
    assert L.fftb_inverse(p._h, vp(d_c.data_ptr()), vp(buf.data_ptr() + 16), 1, None) == fb.FFTB_EINVAL
    assert L.fftb_forward(p._h, vp(buf.data_ptr() + 16), vp(d_c.data_ptr()), 1, None) == fb.FFTB_EINVAL
    assert L.fftb_inverse(p._h, vp(d_c.data_ptr() + 8), vp(buf.data_ptr()), 1, None) == fb.FFTB_EINVAL
    assert L.fftb_inverse(p._h, vp(d_c.data_ptr() + 16), vp(buf.data_ptr() + 32), 1, None) == fb.FFTB_OK
    torch.cuda.synchronize()
    p.destroy()


# ---------------------------------------------------------------------------------------------------------------
# band sharding and host threads on the CUDA path
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,a,dtype,nb", [((128, 128, 128), (32, 32, 32), "c128", 11), ((64, 64, 64), (16, 16, 16), "c128", 9),
                                          ((96, 96, 192), (24, 24, 48), "c64", 6)])
def test_band_shards_are_bit_identical_to_the_unsharded_call(fb, oracle, n, a, dtype, nb):
    """the batch is the only dimension split over GPUs.  Two shards
    (sharding.band_range, world 2) run through two plans on two streams of one device: the concatenation equals the
    unsharded fftb_inverse / fftb_apply_vloc result bit for bit, and the oracle within tolerance."""
    w = _w(n, a, dtype=dtype, batch=nb)
    whole = fb.Plan(n, a, batch=nb, dtype=dtype).bind()
    k = whole.points()
    c = wl.coefficients(w, *k)
    v = wl.potential(w)
    d_c, d_v = torch.from_numpy(c).cuda(), torch.from_numpy(v).cuda()
    psi = whole.inverse(d_c)
    hv = whole.apply_vloc(d_c, d_v)
    torch.cuda.synchronize()
    parts_psi, parts_hv, streams, plans = [], [], [], []
    for r in range(2):
        lo, hi = band_range(nb, 2, r)
        pr = fb.Plan(n, a, batch=hi - lo, dtype=dtype).bind()
        s = torch.cuda.Stream()
        s.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(s):
            shard = d_c[lo:hi].clone()  # a fresh allocation: a complex64 slice that starts on an odd band is only 8-byte aligned
            parts_psi.append(pr.inverse(shard, stream=s))
            parts_hv.append(pr.apply_vloc(shard, d_v, stream=s))
        streams.append(s); plans.append(pr)
    for s in streams:
        s.synchronize()
    assert torch.equal(torch.cat(parts_psi), psi) and torch.equal(torch.cat(parts_hv), hv)
    sample = [0, nb - 1]
    assert _rel(psi[sample].cpu().numpy(), oracle.inverse(n, k, c[sample])) <= w.tol
    assert _rel(hv[sample].cpu().numpy(), oracle.apply_vloc(n, k, c[sample], v, 1.0 / float(np.prod(n)))) <= w.tol
    for pr in plans + [whole]:
        pr.destroy()


@pytest.mark.timeout(300)
def test_two_host_threads_two_plans(fb):
    """Two host threads drive two plans of different pitch through the same kernel instantiations on two streams
    (ctypes releases the GIL during the calls): the launch-side state is per plan or guarded, so every result equals
    the one the same plan produced alone."""
    specs = [((128, 128, 128), (32, 32, 32), 6), ((128, 128, 128), (20, 27, 13), 5), ((64, 64, 64), (16, 16, 16), 7), ((64, 64, 64), (9, 12, 16), 4)]
    jobs = []
    for i, (n, a, nb) in enumerate(specs):
        w = _w(n, a, batch=nb)
        p = fb.Plan(n, a, batch=nb, tuning={"flags": fb.FFTB_TUNE_FUSED} if i == 1 else None).bind()
        d_c = torch.from_numpy(wl.coefficients(w, *p.points())).cuda()
        d_v = torch.from_numpy(wl.potential(w)).cuda()
        ref = (p.inverse(d_c).clone(), p.forward(p.inverse(d_c)).clone(), p.apply_vloc(d_c, d_v).clone())
        jobs.append((p, d_c, d_v, ref))
    torch.cuda.synchronize()
    errors = []

    def run(my):
        try:
            s = torch.cuda.Stream()
            with torch.cuda.stream(s):
                for _ in range(8):
                    for p, d_c, d_v, ref in my:
                        psi = p.inverse(d_c, stream=s)
                        rt = p.forward(psi, stream=s)
                        hv = p.apply_vloc(d_c, d_v, stream=s)
                        s.synchronize()
                        if not (torch.equal(psi, ref[0]) and torch.equal(rt, ref[1]) and torch.equal(hv, ref[2])):
                            errors.append("mismatch")
        except Exception as exc:  # noqa: BLE001
            errors.append(repr(exc))

    th = [threading.Thread(target=run, args=(jobs[0::2],)), threading.Thread(target=run, args=(jobs[1::2],))]
    for t in th:
        t.start()
    for t in th:
        t.join()
    assert not errors, errors[:3]
    for p, *_ in jobs:
        p.destroy()


# ---------------------------------------------------------------------------------------------------------------
# batch-fastest packed arrays (Fig. 8 "b x y z")
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,a,dtype,nb", [((64, 64, 64), (16, 16, 16), "c128", 7), ((128, 128, 128), (32, 32, 32), "c128", 5),
                                          ((96, 96, 192), (24, 24, 48), "c64", 6), ((128, 128, 64), (32, 20, 16), "c64", 37),
                                          ((96, 96, 96), (24, 24, 24), "c128", 1), ((256, 256, 128), (40, 64, 32), "c128", 2)])
def test_batch_fastest_plans_vs_oracle(fb, oracle, n, a, dtype, nb):
    """FFTB_FLAG_BATCH_FASTEST: the packed arrays of every call are [S][nb] (band index fastest); the z passes read and
    write them directly.  Inverse, forward of a generic cuboid and the fused local potential against the oracle's
    results TRANSPOSED, and bit for bit against the band-slowest plan (the arithmetic is the same, only the addresses
    of the packed elements differ).  The input must survive and nothing outside [0, S nb) may be written."""
    w = _w(n, a, dtype=dtype, batch=nb)
    pf = fb.Plan(n, a, batch=nb, dtype=dtype, batch_fastest=True).bind()
    ps = fb.Plan(n, a, batch=nb, dtype=dtype).bind()
    k = ps.points()
    c = wl.coefficients(w, *k)                                       # [nb][S]
    d_c = torch.from_numpy(c).cuda()
    d_ct = torch.from_numpy(np.ascontiguousarray(c.T)).cuda()         # [S][nb]
    psi = pf.inverse(d_ct)
    torch.cuda.synchronize()
    assert torch.equal(psi, ps.inverse(d_c)) and torch.equal(d_ct.cpu(), torch.from_numpy(np.ascontiguousarray(c.T)))
    sample = [0, nb - 1]
    if n[0] <= 128:
        assert _rel(psi[sample].cpu().numpy(), oracle.inverse(n, k, c[sample])) <= w.tol
    g = wl.cuboid(w)
    d_g = torch.from_numpy(g).cuda()
    guard = 4
    buf = torch.full((guard + pf.S * nb + guard,), 777.0 - 555.0j, dtype=pf.torch_complex, device="cuda")
    out = buf[guard:guard + pf.S * nb].view(pf.S, nb)
    pf.forward(d_g, out)
    torch.cuda.synchronize()
    h = buf.cpu().numpy()
    assert (h[:guard] == h[0]).all() and (h[-guard:] == h[0]).all() and h[0] == np.asarray(777.0 - 555.0j, dtype=h.dtype)
    assert torch.equal(out.t().contiguous(), ps.forward(d_g))
    C = float(np.prod(n))
    if n[0] <= 128:
        assert _rel(out.t()[sample].cpu().numpy(), oracle.forward(n, k, g[sample], 1.0 / C)) <= w.tol
    v = wl.potential(w)
    d_v = torch.from_numpy(v).cuda()
    hv = pf.apply_vloc(d_ct, d_v)
    torch.cuda.synchronize()
    assert tuple(hv.shape) == (pf.S, nb) and torch.equal(hv.t().contiguous(), ps.apply_vloc(d_c, d_v))
    if n[0] <= 128:
        assert _rel(hv.t()[sample].cpu().numpy(), oracle.apply_vloc(n, k, c[sample], v, 1.0 / C)) <= w.tol
    pf.destroy(); ps.destroy()


def test_batch_fastest_band_chunks_and_host_calls(fb, oracle):
    """A workspace of two bands makes the library walk a batch-fastest array chunk by chunk (column ranges of [S][nb]),
    and the *_host calls move such an array in one piece."""
    n, a, nb = (64, 64, 64), (16, 16, 16), 7
    w = _w(n, a, batch=nb)
    p = fb.Plan(n, a, batch=nb, batch_fastest=True, tuning={"workspace_bytes": 2 * 64 * 800 * 16 * 2}).bind(host_staging=True)
    assert p.info["chunk_bands"] < nb
    k = p.points()
    c = wl.coefficients(w, *k)
    ct = np.ascontiguousarray(c.T)
    psi = p.inverse(torch.from_numpy(ct).cuda())
    rt = p.forward(psi)
    torch.cuda.synchronize()
    assert _rel(psi.cpu().numpy(), oracle.inverse(n, k, c)) <= w.tol and _rel(rt.cpu().numpy(), ct) <= w.tol
    h_in = torch.from_numpy(ct).pin_memory()
    h_out = torch.empty_like(h_in).pin_memory()
    v = wl.potential(w)
    p.apply_vloc_host(h_in, h_out, torch.from_numpy(v).cuda())
    torch.cuda.synchronize()
    assert _rel(h_out.numpy().T, oracle.apply_vloc(n, k, c, v, 1.0 / float(np.prod(n)))) <= w.tol
    p.destroy()


# ---------------------------------------------------------------------------------------------------------------
# wider predefined patterns: N1 != N2 and cut-offs beyond N/4
# ---------------------------------------------------------------------------------------------------------------
WIDER = [((32, 64, 32), (8, 16, 8), "c128"), ((64, 32, 96), (16, 8, 24), "c64"), ((64, 128, 96), (16, 32, 24), "c128"),
         ((128, 64, 256), (32, 16, 64), "c64"), ((128, 64, 64), (20, 7, 16), "c128"),
         ((32, 32, 32), (12, 8, 8), "c128"), ((64, 64, 64), (24, 31, 20), "c128"), ((128, 128, 64), (40, 50, 31), "c128"),
         ((64, 64, 128), (16, 16, 60), "c128"), ((32, 32, 32), (12, 8, 8), "c64"), ((64, 64, 256), (24, 31, 100), "c64"),
         ((128, 128, 64), (40, 50, 31), "c64")]


@pytest.mark.parametrize("n,a,dtype", WIDER, ids=[f"{n[0]}x{n[1]}x{n[2]}-a{a[0]}.{a[1]}.{a[2]}-{d}" for n, a, d in WIDER])
def test_rectangular_grids_and_wide_cutoffs_vs_oracle(fb, oracle, n, a, dtype):
    """Grids with N1 != N2 (generic plane kernel, one axis pattern per axis) and cut-offs with N/4 < a < N/2 on some axis
    (full-band axis patterns with the pruned stick map): map bit-exact, inverse / forward / local potential vs the oracle."""
    nb = 3
    w = _w(n, a, dtype=dtype, batch=nb)
    p = fb.Plan(n, a, batch=nb, dtype=dtype).bind()
    k = p.points()
    assert all(np.array_equal(x, y) for x, y in zip(k, oracle.enum_points(n, a)))
    c = wl.coefficients(w, *k)
    d_c = torch.from_numpy(c).cuda()
    d_psi = p.inverse(d_c)
    torch.cuda.synchronize()
    assert _rel(d_psi.cpu().numpy(), oracle.inverse(n, k, c)) <= w.tol
    g = wl.cuboid(w)
    C = float(np.prod(n))
    d_f = p.forward(torch.from_numpy(g).cuda())
    v = wl.potential(w)
    d_o = p.apply_vloc(d_c, torch.from_numpy(v).cuda())
    rt = p.forward(d_psi)
    torch.cuda.synchronize()
    assert _rel(d_f.cpu().numpy(), oracle.forward(n, k, g, 1.0 / C)) <= w.tol
    assert _rel(d_o.cpu().numpy(), oracle.apply_vloc(n, k, c, v, 1.0 / C)) <= w.tol
    assert _rel(rt.cpu().numpy(), c) <= w.tol
    p.destroy()


# ---------------------------------------------------------------------------------------------------------------
# dense arm on the line-pass kernel (fftb_dense.cuh), both precisions
# ---------------------------------------------------------------------------------------------------------------
DENSE = [((64, 64, 64), "c128", {}), ((64, 64, 64), "c64", {}), ((128, 128, 128), "c128", {}), ((128, 128, 128), "c64", {}),
         ((256, 256, 256), "c128", {}), ((256, 256, 256), "c64", {}),
         ((32, 32, 32), "c64", {}), ((32, 32, 64), "c64", {}), ((64, 64, 64), "c64", {"flags": 3}), ((64, 64, 64), "c128", {"flags": 3})]


@pytest.mark.timeout(600)
@pytest.mark.parametrize("n,dtype,tuning", DENSE, ids=[f"{n[0]}x{n[2]}-{d}-{'generic' if t else 'default'}" for n, d, t in DENSE])
def test_dense_arm_vs_oracle(fb, oracle, n, dtype, tuning):
    """FFTB_FLAG_DENSE plans (every point of the cube is a coefficient) against the oracle, whose
    transform is dense anyway: inverse of random coefficients, forward of a generic cuboid, the fused local-potential
    apply, and the round trip.  Cubes of 64, 128, 256 points run the line-pass kernel (three passes per direction, the
    first radix-2 split with data in both halves), the others and `flags = generic` the generic kernels.  256^3: the
    oracle's defining sums at sampled outputs (its full transform of 16.7 M points per band takes too long here)."""
    big = n[0] >= 256
    nb = 1 if big else 2
    w = _w(n, (0, 0, 0), dtype=dtype, batch=nb, number=5)
    p = fb.Plan(n, batch=nb, dtype=dtype, dense=True, tuning=tuning or None).bind()
    assert p.S == n[0] * n[1] * n[2] and p.info["y_residues"] == (1 if not tuning and n[0] == n[2] and n[0] >= 64 else p.info["y_residues"])
    k = p.points()
    c = wl.coefficients(w, *k)
    g = wl.cuboid(w, batch=nb)
    v = wl.potential(w)
    C = float(np.prod(n))
    d_c, d_g, d_v = torch.from_numpy(c).cuda(), torch.from_numpy(g).cuda(), torch.from_numpy(v).cuda()
    d_psi = p.inverse(d_c)
    assert p.last_launches() == (3 if not tuning and n[0] == n[2] and n[0] >= 64 else p.last_launches())
    d_f = p.forward(d_g)
    d_o = p.apply_vloc(d_c, d_v)
    d_rt = p.forward(d_psi)
    torch.cuda.synchronize()
    assert torch.equal(d_c.cpu(), torch.from_numpy(c)) and torch.equal(d_g.cpu(), torch.from_numpy(g))
    assert _rel(d_rt.cpu().numpy(), c) <= w.tol
    if not big:
        assert _rel(d_psi.cpu().numpy(), oracle.inverse(n, k, c)) <= w.tol
        assert _rel(d_f.cpu().numpy(), oracle.forward(n, k, g, 1.0 / C)) <= w.tol
        assert _rel(d_o.cpu().numpy(), oracle.apply_vloc(n, k, c, v, 1.0 / C)) <= w.tol
    else:
        rng = np.random.default_rng(7)
        idx = np.concatenate([[0, 1, int(C) - 1, n[0] * n[1], n[0]], rng.integers(0, int(C), size=11)]).astype(np.int64)
        want = oracle.brute_inverse_at(n, k, c, idx)
        got = d_psi.cpu().numpy().reshape(nb, -1)[:, idx]
        scale = np.linalg.norm(d_psi.cpu().numpy().ravel()) / np.sqrt(C)   # rms magnitude of an output
        assert np.max(np.abs(got - want)) <= w.tol * scale * np.sqrt(np.log2(C))
        wantf = oracle.brute_forward_at(n, k, g, idx, 1.0 / C)
        gotf = d_f.cpu().numpy()[:, idx]
        scalef = np.linalg.norm(d_f.cpu().numpy().ravel()) / np.sqrt(C)
        assert np.max(np.abs(gotf - wantf)) <= w.tol * scalef * np.sqrt(np.log2(C))
        # the local-potential apply against its own two halves (each checked above)
        chk = p.forward((d_psi * d_v.unsqueeze(0)).contiguous())
        assert _rel(d_o.cpu().numpy(), chk.cpu().numpy()) <= w.tol
    p.destroy()


# ---------------------------------------------------------------------------------------------------------------
# explicit stick maps with holes (the offsets array describes any set of z-sticks)
# ---------------------------------------------------------------------------------------------------------------
HOLES = [((64, 64, 64), 13, (1, -2, 3), "c128", {}), ((128, 128, 128), 27, (-3, 4, 2), "c128", {}), ((128, 128, 128), 27, (-3, 4, 2), "c64", {}),
         ((256, 256, 64), 14, (1, -1, 1), "c128", {}), ((32, 32, 96), 6, (1, 1, -9), "c64", {}), ((64, 64, 64), 25, (1, 0, -2), "c128", {}),
         ((128, 128, 128), 27, (-3, 4, 2), "c128", {"flags": 4}), ((64, 64, 64), 13, (1, -2, 3), "c128", {"flags": 3})]


@pytest.mark.timeout(300)
@pytest.mark.parametrize("n,radius,centre,dtype,tuning", HOLES,
                         ids=[f"{n[0]}x{n[2]}-r{r}-{d}-{t.get('flags', 0)}" for n, r, c, d, t in HOLES])
def test_explicit_map_with_holes_vs_oracle(fb, oracle, n, radius, centre, dtype, tuning):
    """A k-point-shifted ball with randomly shortened sticks, out of which the test then removes sticks: single sticks
    and runs of 1 - 40 sticks inside k2 runs, the first stick after a column start, and whole k1 columns (two of them
    neighbours).  The plan fills the holes with zero-length sticks of its own; the caller sees its own map, the packed
    array has no element for them, and inverse / forward / local potential match the oracle's plain definition on the
    point list the TEST expands from the map.  Persistent TMA kernels (64, 128, 256 half-band), generic kernels (32;
    radius 25 on 64: full-band), the fused launch (flags 4)."""
    from test_host_cabi import _shifted_ball_map

    full = _shifted_ball_map(n, radius, centre, trim_seed=11)
    k1f, k2f = full[0], full[1]
    rng = np.random.default_rng(radius)
    keep = np.ones(k1f.size, bool)
    cols = np.unique(k1f)
    for c1 in (cols[2], cols[3], cols[len(cols) // 2]):                      # whole k1 columns, two of them neighbours
        keep[k1f == c1] = False
    for c1 in cols[5:-2:3]:                                                  # holes inside k2 runs
        idx = np.flatnonzero(k1f == c1)
        if idx.size >= 5:
            a = int(rng.integers(1, idx.size - 2))
            b = min(idx.size - 1, a + int(rng.integers(1, 41)))
            keep[idx[a:b]] = False
    sm = tuple(x[keep] for x in full)
    assert sm[0].size < k1f.size - 10
    nb = 3
    p = fb.Plan(n, batch=nb, dtype=dtype, stick_map=sm, tuning=tuning or None).bind()
    if tuning.get("flags") == 4:
        assert p.info["ring_bands"] >= 1
    m = p.get_map()
    for key, ref in zip(("k1", "k2", "k3lo", "len"), sm):
        assert np.array_equal(m[key], ref), key
    rep = np.repeat(np.arange(sm[0].size), sm[3])
    off = np.concatenate([[0], np.cumsum(sm[3])])[:-1]
    k = (sm[0][rep], sm[1][rep], (sm[2][rep] + (np.arange(rep.size) - off[rep])).astype(np.int32))
    assert p.S == rep.size and all(np.array_equal(x, y) for x, y in zip(p.points(), k))
    w = _w(n, (0, 0, 0), dtype=dtype, batch=nb)
    c = wl.coefficients(w, *k)
    g = wl.cuboid(w)
    v = wl.potential(w)
    C = float(np.prod(n))
    d_c = torch.from_numpy(c).cuda()
    d_psi = p.inverse(d_c)
    d_f = p.forward(torch.from_numpy(g).cuda())
    d_o = p.apply_vloc(d_c, torch.from_numpy(v).cuda())
    d_rt = p.forward(d_psi)
    torch.cuda.synchronize()
    assert _rel(d_psi.cpu().numpy(), oracle.inverse(n, k, c)) <= w.tol
    assert _rel(d_f.cpu().numpy(), oracle.forward(n, k, g, 1.0 / C)) <= w.tol
    assert _rel(d_o.cpu().numpy(), oracle.apply_vloc(n, k, c, v, 1.0 / C)) <= w.tol
    assert _rel(d_rt.cpu().numpy(), c) <= w.tol
    p.destroy()
