"""CPU oracle for the FFTB sphere <-> cuboid transform -- TEST INFRASTRUCTURE ONLY.

Thin ctypes/numpy front end to ``fftb_oracle.c`` (see that file's header for the
PAPER.md passages each routine follows).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl
reference`` legs may import this package; the product package
``paper_2406_05577_b200`` never does, and this package never imports it.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "fftb_oracle.c"
_LIB = _HERE / "libfftb_oracle.so"
_lib = None


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (-O2 -fopenmp). Building the checker is not using it."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".tmp{os.getpid()}.so")
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-std=c99", "-fPIC", "-shared", "-o", str(tmp), str(_SRC), "-lm"]
        )
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(str(_LIB))
        _lib.orc_enum_points.restype = ctypes.c_int64
        _lib.orc_stick_map.restype = ctypes.c_int64
    return _lib


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def _i3(v):
    return np.ascontiguousarray(np.asarray(v, dtype=np.int32).reshape(3))


def num_threads() -> int:
    return int(_load().orc_num_threads())


def dft1d(x, sign: int, naive: bool = False):
    """1D DFT of PAPER.md Eq. 2-3; sign=-1 forward, +1 inverse (unnormalised)."""
    x = np.ascontiguousarray(x, dtype=np.complex128)
    y = np.empty_like(x)
    fn = _load().orc_dft1d_naive if naive else _load().orc_dft1d
    rc = fn(ctypes.c_int(x.size), ctypes.c_int(sign), _p(x), _p(y))
    if rc:
        raise ValueError(f"orc_dft1d rc={rc}")
    return y


def enum_points(n, a):
    """Cut-off points in packed order -> (k1, k2, k3) int32 arrays of length S."""
    n, a = _i3(n), _i3(a)
    S = _load().orc_enum_points(_p(n), _p(a), None, None, None)
    if S < 0:
        raise ValueError(f"invalid grid/cutoff n={n} a={a}")
    k = [np.empty(S, dtype=np.int32) for _ in range(3)]
    _load().orc_enum_points(_p(n), _p(a), _p(k[0]), _p(k[1]), _p(k[2]))
    return tuple(k)


def stick_map(n, a):
    """The offset array -> dict(k1, k2, k3lo, len (int32[n_sticks]), off (int64[n_sticks+1]))."""
    n, a = _i3(n), _i3(a)
    ns = _load().orc_stick_map(_p(n), _p(a), None, None, None, None, None)
    if ns < 0:
        raise ValueError(f"orc_stick_map rc={ns}")
    m = {key: np.empty(ns, dtype=np.int32) for key in ("k1", "k2", "k3lo", "len")}
    m["off"] = np.empty(ns + 1, dtype=np.int64)
    _load().orc_stick_map(_p(n), _p(a), _p(m["k1"]), _p(m["k2"]), _p(m["k3lo"]), _p(m["len"]), _p(m["off"]))
    return m


def _prep(n, k, coef):
    n = _i3(n)
    k = [np.ascontiguousarray(x, dtype=np.int32) for x in k]
    coef = np.ascontiguousarray(coef, dtype=np.complex128)  # complex64 inputs are widened, never narrowed
    if coef.ndim == 1:
        coef = coef[None, :]
    assert coef.shape[1] == k[0].size
    return n, k, coef


def inverse(n, k, coef, n_axes: int = 3):
    """Packed sphere coef[nb][S] -> cuboid psi[nb][N3][N2][N1] (unnormalised, +j sign)."""
    n, k, coef = _prep(n, k, coef)
    nb, S = coef.shape
    psi = np.empty((nb, int(n[2]), int(n[1]), int(n[0])), dtype=np.complex128)
    rc = _load().orc_inverse(_p(n), ctypes.c_int64(S), _p(k[0]), _p(k[1]), _p(k[2]), _p(coef), _p(psi),
                             ctypes.c_int(nb), ctypes.c_int(n_axes))
    if rc:
        raise ValueError(f"orc_inverse rc={rc}")
    return psi


def forward(n, k, psi, scale: float = 1.0):
    """Cuboid psi[nb][N3][N2][N1] -> packed sphere coef[nb][S], times scale (-j sign)."""
    n = _i3(n)
    k = [np.ascontiguousarray(x, dtype=np.int32) for x in k]
    psi = np.ascontiguousarray(psi, dtype=np.complex128)
    if psi.ndim == 3:
        psi = psi[None]
    assert psi.shape[1:] == (int(n[2]), int(n[1]), int(n[0]))
    nb, S = psi.shape[0], k[0].size
    coef = np.empty((nb, S), dtype=np.complex128)
    rc = _load().orc_forward(_p(n), ctypes.c_int64(S), _p(k[0]), _p(k[1]), _p(k[2]), _p(psi), _p(coef),
                             ctypes.c_int(nb), ctypes.c_double(scale))
    if rc:
        raise ValueError(f"orc_forward rc={rc}")
    return coef


def apply_vloc(n, k, coef, vloc, scale: float = 1.0):
    """c' = forward(V .* inverse(c)) * scale, V real [N3][N2][N1]."""
    n, k, coef = _prep(n, k, coef)
    nb, S = coef.shape
    vloc = np.ascontiguousarray(vloc, dtype=np.float64)
    assert vloc.shape == (int(n[2]), int(n[1]), int(n[0]))
    out = np.empty_like(coef)
    rc = _load().orc_apply_vloc(_p(n), ctypes.c_int64(S), _p(k[0]), _p(k[1]), _p(k[2]), _p(coef), _p(out),
                                _p(vloc), ctypes.c_int(nb), ctypes.c_double(scale))
    if rc:
        raise ValueError(f"orc_apply_vloc rc={rc}")
    return out


def brute_inverse_at(n, k, coef, idx):
    """The defining sum (Eq. 8) at the listed linear cuboid indices -> out[nb][len(idx)]."""
    n, k, coef = _prep(n, k, coef)
    nb, S = coef.shape
    idx = np.ascontiguousarray(idx, dtype=np.int64)
    out = np.empty((nb, idx.size), dtype=np.complex128)
    _load().orc_brute_inverse_at(_p(n), ctypes.c_int64(S), _p(k[0]), _p(k[1]), _p(k[2]), _p(coef),
                                 ctypes.c_int(nb), _p(idx), ctypes.c_int64(idx.size), _p(out))
    return out


def brute_forward_at(n, k, psi, pidx, scale: float = 1.0):
    """The defining sum (Eq. 3-4) at the listed packed indices -> out[nb][len(pidx)]."""
    n = _i3(n)
    k = [np.ascontiguousarray(x, dtype=np.int32) for x in k]
    psi = np.ascontiguousarray(psi, dtype=np.complex128)
    if psi.ndim == 3:
        psi = psi[None]
    nb = psi.shape[0]
    pidx = np.ascontiguousarray(pidx, dtype=np.int64)
    out = np.empty((nb, pidx.size), dtype=np.complex128)
    _load().orc_brute_forward_at(_p(n), _p(k[0]), _p(k[1]), _p(k[2]), _p(psi), ctypes.c_int(nb), _p(pidx),
                                 ctypes.c_int64(pidx.size), ctypes.c_double(scale), _p(out))
    return out
