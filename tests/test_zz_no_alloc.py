"""fftb_inverse_static (include/fftb.h): the inverse transform for callers that may not allocate device memory -- the
plan's tables and the intermediate A in the library's own `static __device__` array of FFTB_STATIC_SCRATCH_BYTES, no
bind block.  It launches the same kernels as fftb_inverse, so the bar is the strictest one the GPU tests use for two
launch paths of the same arithmetic (fused vs separate launches, tests/test_gpu_round2.py): bit-identical outputs.

This file is named to be collected LAST: the suite runs with pytest -x, and a failure here must not hide other tests.
Every test works in a fresh process (it creates its own plans and buffers) and after the other tests (the static array
then holds whatever earlier calls left, which is what the stale-contents test provokes on purpose)."""
import numpy as np
import pytest

from paper_2406_05577_b200 import workloads as wl

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def fb():
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2406_05577_b200 import binding

    binding.lib()
    return binding


def _w(n, a, dtype="c128", batch=3, dist="uniform", number=0):
    return wl.Workload(number, "t", n, a, dtype, batch, dist, "inv_fwd")


def _inputs(fb, w, **plan_kw):
    """(bound plan for the existing path, unbound plan for the static path, device coefficients)"""
    bound = fb.Plan(w.n, w.cutoff, batch=w.batch, dtype=w.dtype, **plan_kw).bind()
    unbound = fb.Plan(w.n, w.cutoff, batch=w.batch, dtype=w.dtype, **plan_kw)
    assert unbound.mem is None
    c = wl.coefficients(w, *bound.points())
    return bound, unbound, torch.from_numpy(c).cuda()


CASES = [
    # n, cut-off, dtype, bands: persistent TMA kernels (64, 96, 128), generic kernels (32, rectangular, full band, dense),
    # batches smaller and larger than what the array holds at once (128^3 complex128: two bands at a time)
    ((32, 32, 32), (8, 8, 8), "c128", 4, {}),
    ((64, 64, 64), (16, 16, 16), "c128", 5, {}),
    ((64, 64, 64), (16, 16, 16), "c64", 3, {}),
    ((96, 96, 192), (24, 24, 48), "c64", 3, {}),
    ((128, 128, 128), (32, 32, 32), "c128", 5, {}),
    ((128, 128, 128), (32, 32, 32), "c64", 7, {}),
    ((64, 128, 64), (16, 32, 16), "c128", 2, {}),
    ((64, 64, 64), (20, 9, 25), "c128", 2, {}),
    ((32, 32, 32), (0, 0, 0), "c128", 2, {"dense": True}),
]


@pytest.mark.timeout(300)
@pytest.mark.parametrize("n,a,dtype,nb,kw", CASES)
def test_static_inverse_equals_bound_inverse_twice(fb, n, a, dtype, nb, kw):
    """Two calls in a row of the no-allocation entry point, each bit-identical to fftb_inverse of a bound plan; the
    second call starts from the array as the first one left it."""
    w = _w(n, a, dtype=dtype, batch=nb, dist="normal_decay", number=3)
    bound, unbound, d_c = _inputs(fb, w, **kw)
    ref = bound.inverse(d_c)
    out = torch.full(bound.cuboid_shape(nb), float("nan"), dtype=bound.torch_complex, device="cuda")
    for call in range(2):
        out.fill_(float("nan"))
        unbound.inverse_static(d_c, out)
        torch.cuda.synchronize()
        assert torch.equal(out, ref), (call, float((out - ref).abs().max()))
    # a different input through the same array
    d_c2 = torch.flip(d_c, dims=[0]).contiguous() * 0.5
    ref2 = bound.inverse(d_c2)
    unbound.inverse_static(d_c2, out)
    assert torch.equal(out, ref2)
    # and a bound plan may use it as well: its bind block is not touched
    before = bound.mem.clone()
    bound.inverse_static(d_c, out)
    assert torch.equal(out, ref) and torch.equal(bound.mem, before)


@pytest.mark.timeout(300)
def test_static_inverse_matches_the_oracle(fb, oracle):
    """The same bar as the parity tests of the bound path (north_star: relative L2 1e-12 for complex128)."""
    w = wl.WORKLOADS[1]
    _, unbound, d_c = _inputs(fb, w)
    ko = oracle.enum_points(w.n, w.cutoff)
    assert all(np.array_equal(x, y) for x, y in zip(unbound.points(), ko))
    want = oracle.inverse(w.n, ko, d_c.cpu().numpy())
    out = torch.empty(unbound.cuboid_shape(w.batch), dtype=unbound.torch_complex, device="cuda")
    for _ in range(2):
        out.zero_()
        unbound.inverse_static(d_c, out)
        got = out.cpu().numpy()
        err = np.linalg.norm((got - want).ravel()) / np.linalg.norm(want.ravel())
        assert err <= w.tol, err


@pytest.mark.timeout(300)
def test_static_array_is_shared_and_stale_contents_do_not_matter(fb):
    """Plans of different shapes take turns on the one array (same stream): each call rewrites the tables and every
    element of the intermediate it reads, so whatever the previous call left (tables of another grid, another band's
    intermediate) changes nothing."""
    ws = [_w((128, 128, 128), (32, 32, 32), "c128", 3, "normal_decay", 3), _w((64, 64, 64), (16, 16, 16), "c128", 4),
          _w((96, 96, 192), (24, 24, 48), "c64", 2), _w((32, 32, 32), (8, 8, 8), "c64", 4)]
    sets = [_inputs(fb, w) for w in ws]
    refs = [b.inverse(c) for b, _, c in sets]
    outs = [torch.empty_like(r) for r in refs]
    for rnd in range(3):
        order = [0, 1, 2, 3] if rnd % 2 == 0 else [3, 1, 0, 2]
        for i in order:
            sets[i][1].inverse_static(sets[i][2], outs[i])
        torch.cuda.synchronize()
        for i in order:
            assert torch.equal(outs[i], refs[i]), (rnd, i)


@pytest.mark.timeout(300)
def test_static_inverse_makes_no_device_allocation(fb):
    """Free device memory as the driver reports it does not move across calls (the first call has already loaded the
    kernels and looked the array's address up), and the call works on a side stream."""
    w = _w((64, 64, 64), (16, 16, 16), "c128", 4)
    _, unbound, d_c = _inputs(fb, w)
    out = torch.empty(unbound.cuboid_shape(w.batch), dtype=unbound.torch_complex, device="cuda")
    s = torch.cuda.Stream()
    unbound.inverse_static(d_c, out)
    torch.cuda.synchronize()
    ref = out.clone()
    with torch.cuda.stream(s):
        unbound.inverse_static(d_c, out, stream=s)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    with torch.cuda.stream(s):
        for _ in range(20):
            out.zero_()
            unbound.inverse_static(d_c, out, stream=s)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, (free0, free1)
    assert torch.equal(out, ref)


@pytest.mark.timeout(300)
def test_static_inverse_refuses_what_does_not_fit(fb):
    """256^3 complex128 at radius 64: one band of the intermediate is 50 MiB > FFTB_STATIC_SCRATCH_BYTES -> FFTB_ETOOBIG
    with a message that names the limit, nothing enqueued (the output keeps its contents); bad arguments -> FFTB_EINVAL."""
    w = wl.WORKLOADS[5]
    big = fb.Plan(w.n, w.cutoff, batch=1, dtype="c128")
    assert w.n[2] * big.info["pitch"] * 16 > fb.FFTB_STATIC_SCRATCH_BYTES
    d_c = torch.zeros(big.packed_shape(1), dtype=torch.complex128, device="cuda")
    out = torch.full(big.cuboid_shape(1), 7.0, dtype=torch.complex128, device="cuda")
    with pytest.raises(fb.FftbError) as ei:
        big.inverse_static(d_c, out)
    assert ei.value.code == fb.FFTB_ETOOBIG and "FFTB_STATIC_SCRATCH_BYTES" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((out == 7.0).all())
    # the largest configuration of the bench that fits: 128^3 complex128 (one band = 6.3 MiB)
    ok = fb.Plan((128, 128, 128), (32, 32, 32), batch=2, dtype="c128")
    assert 128 * ok.info["pitch"] * 16 < fb.FFTB_STATIC_SCRATCH_BYTES // 2
    small = fb.Plan((32, 32, 32), (8, 8, 8), batch=2, dtype="c128")
    c = torch.zeros(small.packed_shape(2), dtype=torch.complex128, device="cuda")
    o = torch.zeros(small.cuboid_shape(2), dtype=torch.complex128, device="cuda")
    L = fb.lib()
    import ctypes

    vp = ctypes.c_void_p
    assert L.fftb_inverse_static(small._h, vp(c.data_ptr()), vp(o.data_ptr()), 3, None) == fb.FFTB_EINVAL   # nb > batch
    assert L.fftb_inverse_static(small._h, vp(c.data_ptr()), vp(o.data_ptr()), 0, None) == fb.FFTB_EINVAL
    assert L.fftb_inverse_static(small._h, None, vp(o.data_ptr()), 1, None) == fb.FFTB_EINVAL
    assert L.fftb_inverse_static(small._h, vp(c.data_ptr()), vp(o.data_ptr() + 16), 1, None) == fb.FFTB_EINVAL  # 32-byte rule
    assert L.fftb_inverse_static(None, vp(c.data_ptr()), vp(o.data_ptr()), 1, None) == fb.FFTB_EINVAL
