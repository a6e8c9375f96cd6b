"""Pins for the CPU oracle (CPU only).  Each test ties one part of oracle/fftb_oracle.c to
something other than itself: values fixed by mathematics (closed forms, lattice-point
sequences, invariants), the library special case (numpy.fft on the zero-padded cuboid,
PAPER.md:110-112), or the defining sums written out here in numpy for tiny grids.
"""
import os
import zlib

import numpy as np
import pytest

from paper_2406_05577_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")

TINY = [((8, 8, 8), (2, 2, 2)), ((4, 6, 8), (1, 1, 2)), ((6, 6, 12), (1, 1, 3)), ((5, 4, 3), (2, 1, 1))]


def _read_rows(name):
    rows = []
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            line = line.strip()
            if line and not line.startswith("#"):
                rows.append(line.split())
    return rows


def _grid_phase(n, kvec, sign):
    """exp(sign 2 pi j (k1 i1/N1 + k2 i2/N2 + k3 i3/N3)) on the whole grid, shape [N3][N2][N1]."""
    i3, i2, i1 = np.meshgrid(np.arange(n[2]), np.arange(n[1]), np.arange(n[0]), indexing="ij")
    ph = kvec[0] * i1 / n[0] + kvec[1] * i2 / n[1] + kvec[2] * i3 / n[2]
    return np.exp(sign * 2j * np.pi * ph)


def _rel(a, b):
    return np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300)


def _rand_coef(S, nb, seed):
    rng = np.random.default_rng(seed)
    return rng.uniform(-1, 1, (nb, S)) + 1j * rng.uniform(-1, 1, (nb, S))


# ----------------------------------------------------------------------------- enumeration


def test_lattice_counts(oracle):
    """S = ball(r), n_sticks = disc(r): classical sequences (tests/golden/lattice_counts.txt)."""
    for kind, r, count in _read_rows("lattice_counts.txt"):
        r, count = int(r), int(count)
        N = max(4 * r, 4)
        if kind == "ball":
            k = oracle.enum_points((N, N, N), (r, r, r))
            assert len(k[0]) == count
        else:
            if N > 128:  # disc(64) through the stick map of config 5
                m = oracle.stick_map((N, N, N), (r, r, r))
                assert len(m["k1"]) == count
            else:
                m = oracle.stick_map((N, N, 4), (r, r, 0) if r == 0 else (r, r, 1))
                # with a3 = 1 the (k1,k2) projection of the ellipsoid is still the full disc
                assert len(m["k1"]) == count


def test_cfg1_stick_prefix_by_hand(oracle):
    m = oracle.stick_map((32, 32, 32), (8, 8, 8))
    for i, row in enumerate(_read_rows("cfg1_stick_prefix.txt")):
        k1, k2, k3lo, ln, off = map(int, row)
        assert (m["k1"][i], m["k2"][i], m["k3lo"][i], m["len"][i], m["off"][i]) == (k1, k2, k3lo, ln, off)
    # sticks per k1 plane (SURVEY.md 8(c) [derived]); symmetric, 17 occupied k1
    per_k1 = [int(np.sum(m["k1"] == q)) for q in range(-8, 9)]
    assert per_k1 == [1, 7, 11, 13, 13, 15, 15, 15, 17, 15, 15, 15, 13, 13, 11, 7, 1]


def test_packed_index_landmarks(oracle):
    k1, k2, k3 = oracle.enum_points((32, 32, 32), (8, 8, 8))
    idx = {(a, b, c): p for p, (a, b, c) in enumerate(zip(k1.tolist(), k2.tolist(), k3.tolist()))}
    S = len(k1)
    assert S == 2109
    assert idx[(0, 0, 0)] == (S - 1) // 2 == 1054
    assert idx[(8, 0, 0)] == S - 1
    assert idx[(-8, 0, 0)] == 0
    # point symmetry of the packed order: pidx(-k) = S-1-pidx(k)
    for (a, b, c), p in idx.items():
        assert idx[(-a, -b, -c)] == S - 1 - p


@pytest.mark.parametrize("n,a", TINY + [((32, 32, 32), (8, 8, 8)), ((96, 96, 192), (24, 24, 48))])
def test_enumeration_vs_mask(oracle, n, a):
    """Same set and order as a vectorised mask + lexicographic sort (float-free)."""
    k1, k2, k3 = oracle.enum_points(n, a)
    r1 = np.arange(-(n[0] // 2), (n[0] + 1) // 2, dtype=np.int64)
    r2 = np.arange(-(n[1] // 2), (n[1] + 1) // 2, dtype=np.int64)
    r3 = np.arange(-(n[2] // 2), (n[2] + 1) // 2, dtype=np.int64)
    g1, g2, g3 = np.meshgrid(r1, r2, r3, indexing="ij")
    A1, A2, A3 = (int(x) for x in a)
    mask = (g1 * A2 * A3) ** 2 + (g2 * A1 * A3) ** 2 + (g3 * A1 * A2) ** 2 <= (A1 * A2 * A3) ** 2
    assert np.array_equal(k1, g1[mask]) and np.array_equal(k2, g2[mask]) and np.array_equal(k3, g3[mask])


def test_boundary_points_are_inclusive(oracle):
    """Eq. 9 uses '<=': the 6 axis points |k| = r lie exactly on the boundary and are kept."""
    k1, k2, k3 = oracle.enum_points((32, 32, 32), (8, 8, 8))
    on = (k1.astype(np.int64) ** 2 + k2.astype(np.int64) ** 2 + k3.astype(np.int64) ** 2) == 64
    assert int(on.sum()) == 6  # 64 = 8^2+0+0 only (no other representation as 3 squares)


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_stick_map_structure(oracle, cfg):
    w = wl.WORKLOADS[cfg]
    m = oracle.stick_map(w.n, w.cutoff)
    k = oracle.enum_points(w.n, w.cutoff)
    S = len(k[0])
    assert m["off"][0] == 0 and m["off"][-1] == S
    assert np.all(np.diff(m["off"]) == m["len"]) and np.all(m["len"] >= 1)
    assert m["len"].max() == 2 * w.cutoff[2] + 1 and m["len"].min() == 1
    assert len(np.unique(m["k1"])) == 2 * w.cutoff[0] + 1  # n_xocc
    # expanding the map reproduces the point list
    rep = np.repeat(np.arange(len(m["k1"])), m["len"])
    assert np.array_equal(m["k1"][rep], k[0]) and np.array_equal(m["k2"][rep], k[1])
    assert np.array_equal(m["k3lo"][rep] + (np.arange(S) - m["off"][:-1][rep]), k[2])
    # "almost 16 times" more data when fully padded: 48/pi = 15.28 in the limit
    ratio = np.prod(w.n) / S
    assert 15.2 < ratio < 15.6


def test_offset_crc_fixture(oracle):
    for name, n1, n2, n3, a1, a2, a3, S, ns, crc in _read_rows("offset_crc32.txt"):
        m = oracle.stick_map((int(n1), int(n2), int(n3)), (int(a1), int(a2), int(a3)))
        assert int(m["off"][-1]) == int(S) and len(m["k1"]) == int(ns)
        assert f"{zlib.crc32(m['off'].astype('<i8').tobytes()) & 0xFFFFFFFF:08x}" == crc


def test_invalid_cutoff_rejected(oracle):
    with pytest.raises(ValueError):
        oracle.enum_points((32, 32, 32), (16, 8, 8))  # 2a >= N would alias (R9)
    with pytest.raises(ValueError):
        oracle.enum_points((32, 32, 32), (8, -1, 8))


# ----------------------------------------------------------------------------- 1D building block


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 8, 12, 16, 32, 64, 96, 128, 192, 256])
def test_dft1d_definition_and_library(oracle, n):
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    l, k = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    for sign in (-1, +1):
        W = np.exp(sign * 2j * np.pi * ((l * k) % n) / n)  # DFT_n = [w^{lk}], Eq. 3
        ref = W @ x
        assert _rel(oracle.dft1d(x, sign), ref) < 1e-13
        assert _rel(oracle.dft1d(x, sign, naive=True), ref) < 1e-13
    assert _rel(oracle.dft1d(x, -1), np.fft.fft(x)) < 1e-14
    assert _rel(oracle.dft1d(x, +1), np.fft.ifft(x) * n) < 1e-14


def test_dft1d_sign_convention(oracle):
    """Forward uses w_n = exp(-j 2 pi / n): a unit impulse at index 1 maps to w^l."""
    n = 8
    x = np.zeros(n, complex)
    x[1] = 1
    assert np.allclose(oracle.dft1d(x, -1), np.exp(-2j * np.pi * np.arange(n) / n), atol=1e-15)
    assert np.allclose(oracle.dft1d(x, +1), np.exp(+2j * np.pi * np.arange(n) / n), atol=1e-15)


# ----------------------------------------------------------------------------- inverse


@pytest.mark.parametrize("n,a", TINY)
def test_inverse_brute_force_numpy(oracle, n, a):
    """psi[i] = sum_p c[p] exp(+2 pi j k(p).i/N) written out in numpy (Eq. 8)."""
    k = oracle.enum_points(n, a)
    c = _rand_coef(len(k[0]), 2, 11)
    ref = np.zeros((2, n[2], n[1], n[0]), complex)
    for p in range(len(k[0])):
        ph = _grid_phase(n, (k[0][p], k[1][p], k[2][p]), +1)
        ref += c[:, p, None, None, None] * ph[None]
    psi = oracle.inverse(n, k, c)
    assert _rel(psi, ref) < 1e-14
    idx = np.arange(np.prod(n))
    got = oracle.brute_inverse_at(n, k, c, idx).reshape(ref.shape)
    assert _rel(got, ref) < 1e-14


@pytest.mark.parametrize("n,a", TINY + [((32, 32, 32), (8, 8, 8)), ((24, 12, 48), (6, 3, 12))])
def test_inverse_is_library_ifftn_of_padded_cube(oracle, n, a):
    """zero-pad the sphere into the cuboid, off-the-shelf 3D FFT."""
    k = oracle.enum_points(n, a)
    c = _rand_coef(len(k[0]), 2, 5)
    cube = np.zeros((2, n[2], n[1], n[0]), complex)
    cube[:, k[2] % n[2], k[1] % n[1], k[0] % n[0]] = c
    C = np.prod(n)
    assert _rel(oracle.inverse(n, k, c), np.fft.ifftn(cube, axes=(1, 2, 3)) * C) < 1e-14
    # stage outputs: z only, then z+y
    assert _rel(oracle.inverse(n, k, c, n_axes=1), np.fft.ifft(cube, axis=1) * n[2]) < 1e-14
    assert _rel(oracle.inverse(n, k, c, n_axes=2), np.fft.ifftn(cube, axes=(1, 2)) * n[2] * n[1]) < 1e-14
    assert _rel(oracle.inverse(n, k, c, n_axes=0), cube) == 0.0


def test_inverse_closed_forms(oracle):
    n, a = (32, 32, 32), (8, 8, 8)
    k = oracle.enum_points(n, a)
    S = len(k[0])
    # impulse at k = 0 -> all-ones cuboid
    c = np.zeros((1, S), complex)
    c[0, (S - 1) // 2] = 1
    assert np.abs(oracle.inverse(n, k, c) - 1).max() < 1e-13
    # single plane wave (also a negative-frequency one: exercises the wrap-around, reading R3)
    for p in (0, 1222, 77, S - 1):
        c = np.zeros((1, S), complex)
        c[0, p] = 2 - 0.5j
        ref = (2 - 0.5j) * _grid_phase(n, (k[0][p], k[1][p], k[2][p]), +1)
        assert np.abs(oracle.inverse(n, k, c)[0] - ref).max() < 1e-13


def test_inverse_parseval_and_linearity(oracle):
    n, a = (16, 12, 20), (4, 3, 5)
    k = oracle.enum_points(n, a)
    c = _rand_coef(len(k[0]), 3, 9)
    psi = oracle.inverse(n, k, c)
    C = np.prod(n)
    for b in range(3):  # sum |psi|^2 = C sum |c|^2
        assert abs(np.sum(np.abs(psi[b]) ** 2) - C * np.sum(np.abs(c[b]) ** 2)) < 1e-10 * C
    comb = (0.3 - 2j) * c[0] + 1.7 * c[1]
    assert _rel(oracle.inverse(n, k, comb)[0], (0.3 - 2j) * psi[0] + 1.7 * psi[1]) < 1e-14


# ----------------------------------------------------------------------------- forward


@pytest.mark.parametrize("n,a", TINY)
def test_forward_brute_force_numpy(oracle, n, a):
    """c[p] = s sum_i psi[i] exp(-2 pi j k(p).i/N) written out in numpy (Eq. 3-4)."""
    k = oracle.enum_points(n, a)
    rng = np.random.default_rng(3)
    psi = rng.uniform(-1, 1, (2, n[2], n[1], n[0])) + 1j * rng.uniform(-1, 1, (2, n[2], n[1], n[0]))
    s = 0.37
    ref = np.stack([
        s * np.array([np.sum(psi[b] * _grid_phase(n, (k[0][p], k[1][p], k[2][p]), -1)) for p in range(len(k[0]))])
        for b in range(2)])
    assert _rel(oracle.forward(n, k, psi, s), ref) < 1e-14
    got = oracle.brute_forward_at(n, k, psi, np.arange(len(k[0])), s)
    assert _rel(got, ref) < 1e-14


def test_forward_is_library_fftn_gathered(oracle):
    n, a = (24, 12, 48), (6, 3, 12)
    k = oracle.enum_points(n, a)
    psi = wl.cuboid(wl.Workload(0, "t", n, a, "c128", 2, "uniform", "inv_fwd"))
    full = np.fft.fftn(psi, axes=(1, 2, 3))
    ref = full[:, k[2] % n[2], k[1] % n[1], k[0] % n[0]]
    assert _rel(oracle.forward(n, k, psi), ref) < 1e-14


def test_forward_closed_forms(oracle):
    n, a = (16, 16, 16), (4, 4, 4)
    k = oracle.enum_points(n, a)
    S, C = len(k[0]), np.prod(n)
    i0 = (3, 14, 7)  # (i1, i2, i3)
    psi = np.zeros((1, n[2], n[1], n[0]), complex)
    psi[0, i0[2], i0[1], i0[0]] = 1
    s = 1.0 / C
    ref = s * np.exp(-2j * np.pi * (k[0] * i0[0] / n[0] + k[1] * i0[1] / n[1] + k[2] * i0[2] / n[2]))
    assert np.abs(oracle.forward(n, k, psi, s)[0] - ref).max() < 1e-15
    # constant cuboid -> only k = 0
    c = oracle.forward(n, k, np.full((1, n[2], n[1], n[0]), 2.5 + 0j), s)[0]
    assert abs(c[(S - 1) // 2] - 2.5) < 1e-14
    c[(S - 1) // 2] = 0
    assert np.abs(c).max() < 1e-14


@pytest.mark.parametrize("n,a", [((32, 32, 32), (8, 8, 8)), ((12, 24, 48), (3, 6, 12))])
def test_round_trip_and_projection(oracle, n, a):
    k = oracle.enum_points(n, a)
    C = np.prod(n)
    c = _rand_coef(len(k[0]), 2, 21)
    psi = oracle.inverse(n, k, c)
    assert _rel(oracle.forward(n, k, psi, 1.0), C * c) < 1e-14       # scale NONE: forward(inverse(c)) = C c
    assert _rel(oracle.forward(n, k, psi, 1.0 / C), c) < 1e-14       # scale FORWARD: identity on the sphere
    # inverse(forward(.))/C is a projection: applying it twice = once
    w = wl.Workload(0, "t", n, a, "c128", 1, "uniform", "inv_fwd")
    g = wl.cuboid(w)
    p1 = oracle.inverse(n, k, oracle.forward(n, k, g, 1.0 / C))
    p2 = oracle.inverse(n, k, oracle.forward(n, k, p1, 1.0 / C))
    assert _rel(p2, p1) < 1e-14
    assert _rel(p1, g) > 0.5  # and it is not the identity (g is not band-limited)


# ----------------------------------------------------------------------------- vloc


def test_vloc_constant_and_cosine(oracle):
    n, a = (8, 8, 8), (2, 2, 2)
    k = oracle.enum_points(n, a)
    S, C = len(k[0]), np.prod(n)
    c = _rand_coef(S, 2, 4)
    v = np.full((n[2], n[1], n[0]), 0.75)
    assert _rel(oracle.apply_vloc(n, k, c, v, 1.0 / C), 0.75 * c) < 1e-14
    # V = cos(2 pi m.i/N), m = (1,0,0): c'(q) = (c(q-m) + c(q+m))/2 with c = 0 outside the cut-off
    for m in ((1, 0, 0), (0, 1, 0), (0, 0, 1), (1, 1, 0)):
        v = np.real(_grid_phase(n, m, +1))
        idx = {(x, y, z): p for p, (x, y, z) in enumerate(zip(k[0].tolist(), k[1].tolist(), k[2].tolist()))}
        ref = np.zeros_like(c)
        for (x, y, z), p in idx.items():
            for sg in (+1, -1):
                q = idx.get((x - sg * m[0], y - sg * m[1], z - sg * m[2]))
                if q is not None:
                    ref[:, p] += 0.5 * c[:, q]
        assert _rel(oracle.apply_vloc(n, k, c, v, 1.0 / C), ref) < 1e-14


def test_vloc_hermitian(oracle):
    n, a = (12, 8, 16), (3, 2, 4)
    k = oracle.enum_points(n, a)
    S, C = len(k[0]), np.prod(n)
    c, d = _rand_coef(S, 1, 1), _rand_coef(S, 1, 2)
    v = np.random.default_rng(0).uniform(0, 1, (n[2], n[1], n[0]))
    Hc, Hd = oracle.apply_vloc(n, k, c, v, 1.0 / C), oracle.apply_vloc(n, k, d, v, 1.0 / C)
    assert abs(np.vdot(d, Hc) - np.conj(np.vdot(c, Hd))) < 1e-12


# ----------------------------------------------------------------------------- workloads


def test_workload_generators_are_seeded():
    w = wl.WORKLOADS[1]
    k = (np.zeros(5, np.int32),) * 3
    a, b = wl.coefficients(w, *k), wl.coefficients(w, *k)
    assert np.array_equal(a, b) and a.shape == (4, 5) and a.dtype == np.complex128
    assert np.all(np.abs(a.real) <= 1) and np.all(np.abs(a.imag) <= 1)
    w4 = wl.WORKLOADS[4]
    assert wl.coefficients(w4, *k).dtype == np.complex64 and wl.potential(w4).dtype == np.float32
    v = wl.potential(wl.WORKLOADS[2])
    assert v.shape == (64, 64, 64) and v.min() >= 0 and v.max() < 1
    # config 3: N(0,1)/(1+|k|^2)
    k3 = (np.array([0, 1, 2], np.int32), np.array([0, 0, 2], np.int32), np.array([0, 0, 1], np.int32))
    c3 = wl.coefficients(wl.WORKLOADS[3], *k3, batch=2000)
    sd = c3.real.std(axis=0)
    assert np.allclose(sd, [1.0, 0.5, 0.1], rtol=0.1)
