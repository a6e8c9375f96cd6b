"""CPU-only tests of the C-ABI library: it loads, exports every symbol include/fftb.h declares,
the host plan builder reproduces the oracle's stick map bit for bit, and the error paths return
codes instead of throwing.  No kernel is launched here."""
import ctypes
import os
import re

import numpy as np
import pytest

from paper_2406_05577_b200 import binding as fb
from paper_2406_05577_b200 import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    from paper_2406_05577_b200.build import build

    build()


def test_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "fftb.h")).read()
    declared = set(re.findall(r"\b(fftb_[a-z_]+)\s*\(", hdr))
    assert declared == set(fb.SYMBOLS)
    L = ctypes.CDLL(str(fb._LIBPATH))
    for s in declared:
        assert hasattr(L, s), s


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_stick_map_bit_exact_vs_oracle(oracle, cfg):
    w = wl.WORKLOADS[cfg]
    p = fb.Plan(w.n, w.cutoff, batch=w.batch, dtype=w.dtype)
    m, o = p.get_map(), oracle.stick_map(w.n, w.cutoff)
    for key in ("k1", "k2", "k3lo", "len", "off"):
        assert m[key].dtype == o[key].dtype and np.array_equal(m[key], o[key]), key
    assert p.info["n_points"] == int(o["off"][-1]) and p.info["n_sticks"] == len(o["k1"])
    assert p.info["n_xocc"] == 2 * w.cutoff[0] + 1
    k = oracle.enum_points(w.n, w.cutoff)
    pk = p.points()
    assert all(np.array_equal(a, b) for a, b in zip(pk, k))
    elem = 16 if w.dtype == "c128" else 8
    assert p.info["min_bytes_per_band_dir"] == (p.S + int(np.prod(w.n))) * elem
    p.destroy()


def test_smaller_cutoffs_and_ellipsoids_vs_oracle(oracle):
    for n, a in [((32, 32, 64), (5, 7, 16)), ((64, 64, 32), (16, 3, 0)), ((128, 128, 96), (1, 32, 24)),
                 ((32, 32, 32), (0, 0, 0))]:
        p = fb.Plan(n, a)
        m, o = p.get_map(), oracle.stick_map(n, a)
        for key in ("k1", "k2", "k3lo", "len", "off"):
            assert np.array_equal(m[key], o[key]), (n, a, key)


def test_dense_plan_map():
    p = fb.Plan((32, 32, 64), dense=True)
    m = p.get_map()
    assert p.S == 32 * 32 * 64 and p.info["n_sticks"] == 1024 and p.info["n_xocc"] == 32
    assert np.all(m["len"] == 64) and np.all(m["k3lo"] == -32)
    assert m["k1"][0] == -16 and m["k2"][0] == -16 and m["k1"][-1] == 15 and m["k2"][33] == -15


def _create_rc(n, a, batch=1, dtype=fb.FFTB_C128, scale=fb.FFTB_SCALE_FORWARD, flags=0):
    d = fb.PlanDesc()
    d.n[:] = n
    d.cutoff[:] = a
    d.batch, d.dtype, d.scale, d.flags = batch, dtype, scale, flags
    h = ctypes.c_void_p()
    rc = fb.lib().fftb_plan_create(ctypes.byref(h), ctypes.byref(d))
    if rc == 0:
        fb.lib().fftb_plan_destroy(h)
    return rc


def test_error_paths():
    L = fb.lib()
    assert _create_rc((32, 32, 32), (8, 8, 8)) == fb.FFTB_OK
    assert _create_rc((32, 32, 32), (16, 8, 8)) == fb.FFTB_EINVAL        # 2a >= N aliases (R9)
    assert _create_rc((32, 32, 32), (8, -1, 8)) == fb.FFTB_EINVAL
    assert _create_rc((0, 32, 32), (8, 8, 8)) == fb.FFTB_EINVAL
    assert _create_rc((32, 32, 32), (8, 8, 8), batch=0) == fb.FFTB_EINVAL
    assert _create_rc((32, 32, 32), (8, 8, 8), dtype=7) == fb.FFTB_EINVAL
    assert _create_rc((32, 32, 32), (8, 8, 8), flags=4) == fb.FFTB_EINVAL
    assert _create_rc((64, 64, 64), (16, 16, 16), flags=3) == fb.FFTB_EINVAL       # dense and batch-fastest together
    assert _create_rc((64, 64, 64), (16, 16, 16), flags=2) == fb.FFTB_OK
    assert _create_rc((32, 32, 32), (8, 8, 8), flags=2) == fb.FFTB_EUNSUPPORTED   # no persistent z pass to fold the transposition into
    assert _create_rc((256, 256, 256), (64, 64, 64), flags=2) == fb.FFTB_EUNSUPPORTED
    # outside the predefined patterns
    assert _create_rc((40, 40, 40), (8, 8, 8)) == fb.FFTB_EUNSUPPORTED
    assert _create_rc((32, 64, 32), (8, 8, 8)) == fb.FFTB_OK              # N1 != N2: one of the predefined pairs
    assert _create_rc((96, 64, 32), (8, 8, 8)) == fb.FFTB_EUNSUPPORTED    # ... this one is not
    assert _create_rc((32, 32, 32), (12, 8, 8)) == fb.FFTB_OK             # a > N/4: full-band axis patterns
    assert _create_rc((32, 32, 32), (12, 8, 8), dtype=fb.FFTB_C64) == fb.FFTB_OK
    assert _create_rc((64, 64, 64), (0, 0, 0), dtype=fb.FFTB_C64, flags=1) == fb.FFTB_OK    # dense, either precision
    assert _create_rc((32, 32, 64), (0, 0, 0), dtype=fb.FFTB_C64, flags=1) == fb.FFTB_OK
    assert _create_rc((96, 96, 96), (30, 8, 8)) == fb.FFTB_EUNSUPPORTED   # no full-band pattern of length 96
    assert L.fftb_plan_create(None, None) == fb.FFTB_EINVAL
    assert L.fftb_plan_destroy(None) == fb.FFTB_EINVAL
    assert L.fftb_plan_info_get(None, None) == fb.FFTB_EINVAL
    # execute before bind
    p = fb.Plan((32, 32, 32), (8, 8, 8))
    buf = ctypes.create_string_buffer(64)
    a = ctypes.c_void_p((ctypes.addressof(buf) + 15) // 16 * 16)
    assert L.fftb_inverse(p._h, a, a, 1, None) == fb.FFTB_ESTATE
    assert L.fftb_forward(p._h, None, a, 1, None) == fb.FFTB_EINVAL
    assert L.fftb_plan_bind(p._h, None, 0, None) == fb.FFTB_EINVAL
    assert fb.strerror(fb.FFTB_EUNSUPPORTED).startswith("description outside")
    assert fb.strerror(-99) == "unknown fftb status"


def test_missing_library_fails_loudly(monkeypatch, tmp_path):
    monkeypatch.setattr(fb, "_lib", None)
    monkeypatch.setattr(fb, "_LIBPATH", tmp_path / "nope.so")
    with pytest.raises(ImportError, match="no CPU fallback"):
        fb.lib()


def _shifted_ball_map(n, radius, centre, trim_seed=None):
    """Sticks of the ball |k - centre| <= radius (a k-point-shifted sphere), written out in numpy as
    mask + sort (independent of both the plan builder and the oracle's cut-off enumeration); with
    trim_seed the sticks are shortened at random, so the map is no cut-off of any kind."""
    r = radius + max(abs(c) for c in centre)
    g = np.arange(-r, r + 1)
    k1, k2, k3 = np.meshgrid(g, g, g, indexing="ij")
    inside = (k1 - centre[0]) ** 2 + (k2 - centre[1]) ** 2 + (k3 - centre[2]) ** 2 <= radius ** 2
    cols = inside.any(axis=2)
    m1, m2 = k1[:, :, 0][cols], k2[:, :, 0][cols]
    lo = np.array([g[inside[a + r, b + r]].min() for a, b in zip(m1, m2)])
    hi = np.array([g[inside[a + r, b + r]].max() for a, b in zip(m1, m2)])
    if trim_seed is not None:
        rng = np.random.default_rng(trim_seed)
        cut_lo = rng.integers(0, 3, size=lo.size)
        cut_hi = rng.integers(0, 3, size=lo.size)
        lo2, hi2 = lo + cut_lo, hi - cut_hi
        keep = lo2 <= hi2
        lo, hi = np.where(keep, lo2, lo), np.where(keep, hi2, hi)
    return m1.astype(np.int32), m2.astype(np.int32), lo.astype(np.int32), (hi - lo + 1).astype(np.int32)


def test_explicit_stick_map_round_trip_and_errors():
    """fftb_plan_create_explicit: the map given is the map kept, bit for bit;
    maps outside the predefined patterns are refused with a code."""
    n = (64, 64, 64)
    sm = _shifted_ball_map(n, 11, (2, -3, 4), trim_seed=7)
    p = fb.Plan(n, batch=2, stick_map=sm)
    m = p.get_map()
    for key, ref in zip(("k1", "k2", "k3lo", "len"), sm):
        assert np.array_equal(m[key], ref), key
    assert np.array_equal(m["off"], np.concatenate([[0], np.cumsum(sm[3])]))
    assert p.S == int(sm[3].sum()) and p.info["n_sticks"] == sm[0].size
    p.destroy()
    k1, k2, lo, ln = [x.copy() for x in sm]
    with pytest.raises(fb.FftbError) as e:      # not ascending
        fb.Plan(n, stick_map=(k1[::-1].copy(), k2[::-1].copy(), lo[::-1].copy(), ln[::-1].copy()))
    assert e.value.code == fb.FFTB_EINVAL
    bad = ln.copy(); bad[3] = 0
    with pytest.raises(fb.FftbError) as e:      # empty stick
        fb.Plan(n, stick_map=(k1, k2, lo, bad))
    assert e.value.code == fb.FFTB_EINVAL
    far = lo.copy(); far[0] = 40
    with pytest.raises(fb.FftbError) as e:      # outside [-N/2, N/2)
        fb.Plan(n, stick_map=(k1, k2, far, ln))
    assert e.value.code == fb.FFTB_EINVAL
    wide = ln.copy(); wide[0] = 17 - lo[0] + 1
    fb.Plan(n, stick_map=(k1, k2, lo, wide)).destroy()   # beyond the half band |k| <= N/4: full-band patterns, either precision
    fb.Plan(n, stick_map=(k1, k2, lo, wide), dtype="c64").destroy()
    # holes (a missing stick inside a k2 run, a missing k1 column): accepted, filled by the plan with zero-length sticks
    # of its own that the caller never sees -- the map read back is the map given
    hole = np.ones(k1.size, bool)
    hole[np.flatnonzero(k1 == k1[k1.size // 2])[1]] = False
    hole[k1 == k1[0] + 2] = False
    hm = (k1[hole], k2[hole], lo[hole], ln[hole])
    ph = fb.Plan(n, batch=2, stick_map=hm)
    mh = ph.get_map()
    for key, ref in zip(("k1", "k2", "k3lo", "len"), hm):
        assert np.array_equal(mh[key], ref), key
    assert np.array_equal(mh["off"], np.concatenate([[0], np.cumsum(hm[3])]))
    assert ph.S == int(hm[3].sum()) and ph.info["n_sticks"] == hm[0].size and ph.info["pitch"] >= hm[0].size + 2
    ph.destroy()
    with pytest.raises(fb.FftbError) as e:      # dense + explicit
        fb.Plan(n, stick_map=sm, dense=True)
    assert e.value.code == fb.FFTB_EINVAL
