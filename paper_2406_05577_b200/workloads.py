"""Seeded synthetic workloads shared by the oracle tests and the CUDA path.

This module holds NO arithmetic of the method (no transform, no cut-off test, no
stick map): it only names the five BASELINE.json configurations and draws their
random inputs.  The frequency vectors a generator needs (config 3 scales each
coefficient by 1/(1+|k|^2)) are passed in by the caller, who takes them from
whichever side it is exercising (oracle.enum_points or fftb_plan_get_map).

Recipe: numpy default_rng (PCG64),
seed 1000 + config number for coefficients and 2000 + config number for V(r);
draw order = all real parts of the [Nb][S] array, then all imaginary parts;
complex64 inputs are drawn in double and rounded once to float.  The paper's own
workload is synthetic too (256^3 grid, diameter-128 sphere, batch 256,
PAPER.md:239); these configs are shaped like it (cut-off radius N/4, i.e. a cube
of width twice the sphere diameter).
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class Workload:
    number: int          # 1-based config number (BASELINE.json configs[number-1])
    name: str
    n: tuple             # (N1, N2, N3) = (x fastest, y, z stick axis)
    cutoff: tuple        # integer semi-axes (a1, a2, a3) in index units
    dtype: str           # "c128" | "c64"
    batch: int
    dist: str            # "uniform" | "normal_decay"
    op: str              # "inv_fwd" | "vloc" | "inv_fwd_pruned_vs_dense"

    @property
    def complex_dtype(self):
        return np.complex128 if self.dtype == "c128" else np.complex64

    @property
    def real_dtype(self):
        return np.float64 if self.dtype == "c128" else np.float32

    @property
    def tol(self) -> float:
        """north_star's parity bar: relative L2 error against the oracle."""
        return 1e-12 if self.dtype == "c128" else 1e-5


WORKLOADS = {
    1: Workload(1, "32^3 c128 x4 r=8 inv+fwd", (32, 32, 32), (8, 8, 8), "c128", 4, "uniform", "inv_fwd"),
    2: Workload(2, "64^3 c128 x64 r=16 vloc", (64, 64, 64), (16, 16, 16), "c128", 64, "uniform", "vloc"),
    3: Workload(3, "128^3 c128 x128 r=32 inv+fwd", (128, 128, 128), (32, 32, 32), "c128", 128,
                "normal_decay", "inv_fwd"),
    4: Workload(4, "96x96x192 c64 x64 ellipsoid(24,24,48) vloc", (96, 96, 192), (24, 24, 48), "c64", 64,
                "uniform", "vloc"),
    5: Workload(5, "256^3 c128 x8 r=64 inv+fwd pruned vs dense", (256, 256, 256), (64, 64, 64), "c128", 8,
                "uniform", "inv_fwd_pruned_vs_dense"),
}


def coefficients(w: Workload, k1, k2, k3, batch: int | None = None, seed: int | None = None):
    """Packed sphere coefficients [batch][S] for workload `w` (host numpy array).

    k1, k2, k3: the packed-order frequency vectors (length S), supplied by the caller.
    """
    nb = w.batch if batch is None else batch
    S = len(k1)
    rng = np.random.default_rng(1000 + w.number if seed is None else seed)
    if w.dist == "uniform":
        re = rng.uniform(-1.0, 1.0, size=(nb, S))
        im = rng.uniform(-1.0, 1.0, size=(nb, S))
    elif w.dist == "normal_decay":
        re = rng.standard_normal(size=(nb, S))
        im = rng.standard_normal(size=(nb, S))
        ksq = (np.asarray(k1, dtype=np.float64) ** 2 + np.asarray(k2, dtype=np.float64) ** 2
               + np.asarray(k3, dtype=np.float64) ** 2)
        decay = 1.0 / (1.0 + ksq)
        re *= decay
        im *= decay
    else:
        raise ValueError(w.dist)
    c = re + 1j * im
    return np.ascontiguousarray(c.astype(w.complex_dtype))


def potential(w: Workload, seed: int | None = None):
    """Real local potential V[N3][N2][N1], iid uniform[0,1), in the workload's real precision."""
    rng = np.random.default_rng(2000 + w.number if seed is None else seed)
    v = rng.uniform(0.0, 1.0, size=(w.n[2], w.n[1], w.n[0]))
    return np.ascontiguousarray(v.astype(w.real_dtype))


def cuboid(w: Workload, batch: int | None = None, seed: int = 3000):
    """A generic (not band-limited) real-space cuboid [batch][N3][N2][N1], re/im iid uniform[-1,1)."""
    nb = w.batch if batch is None else batch
    rng = np.random.default_rng(seed + w.number)
    shape = (nb, w.n[2], w.n[1], w.n[0])
    c = rng.uniform(-1.0, 1.0, size=shape) + 1j * rng.uniform(-1.0, 1.0, size=shape)
    return np.ascontiguousarray(c.astype(w.complex_dtype))
