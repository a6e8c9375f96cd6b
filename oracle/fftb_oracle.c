/*
 * fftb_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, double-precision CPU oracle for the sphere <-> cuboid batched 3D
 * complex FFT of arXiv 2406.05577 (FFTB), written from the paper's definitions
 * only.  It shares no code, header, table or constant with the CUDA path under
 * paper_2406_05577_b200/csrc and neither imports the other.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load it.
 *
 * What it computes (PAPER.md line numbers, section in brackets):
 *   - 1D DFT  y = DFT_n x,  DFT_n = [w_n^{lk}],  w_n = exp(-j 2 pi / n)
 *     (Eq. 2-3 [2.1]); that is the FORWARD sign.
 *   - 3D DFT as three batches of 1D DFTs, one per axis, over every line of the
 *     full cuboid (pencil-pencil-pencil, Eq. 6-7 [2.1]);
 *     column-major storage, n0 = x fastest, n2 = z slowest.
 *   - plane-wave expansion psi(r) = sum_g c(g) exp(+j g r) (Eq. 8
 *     [2.2]); that is the INVERSE sign (frequency -> real space).
 *   - cut-off: only g with 1/2 |g|^2 <= E_cut are kept (PAPER.md:100-104,
 *     Eq. 9), inclusive; here an axis-aligned ellipsoid with integer semi-axes
 *     (a1,a2,a3) in index units, tested in exact integers (reading R4).
 *   - the sphere is zero-padded into the full cuboid and the 3D transform is
 *     applied to the entire cube (PAPER.md:110-112 [2.2]).  The paper states
 *     the staged-padding route computes the same transform, so this plain
 *     definition is what the CUDA path must reproduce up to rounding.
 *   - the offset array: project the sphere on the xy-plane, x and y dense, only
 *     z compressed, CSR-like, one array for all bands (Fig. 7,
 *     183-185 [3.3]).
 *   - batching Psi = [psi_0 | ... | psi_{Nb-1}] (Eq. 10).
 *
 * Algorithm, per band (BASELINE.json north_star fixes the style): zero a full
 * double-complex cuboid, scatter c[p] to (k mod N), run a 1D transform along
 * each axis over EVERY line (recursive radix-2 when the length is a power of
 * two, the O(n^2) definition with twiddle index (l*k) mod n otherwise), and
 * for forward gather the sphere entries and scale.  No blocking, fusion,
 * pruning or reordering.
 *
 * Pins: see tests/test_oracle_pins.py (closed forms, lattice counts, CRCs,
 * numpy.fft special case, brute force below).  Nothing here is "parity
 * unpinned".
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double _Complex cplx;

static const double ORC_2PI = 6.283185307179586476925286766559;

/* ------------------------------------------------------------------------ */
/* 1D transforms (Eq. 2-3).  sign = -1 forward, +1 inverse.  */
/* ------------------------------------------------------------------------ */

/* root of unity exp(sign * j * 2 pi * num / den), num already reduced mod den */
static cplx orc_root(int64_t num, int64_t den, int sign)
{
    double ang = ORC_2PI * (double)num / (double)den;
    return cos(ang) + I * (sign * sin(ang));
}

/* O(n^2) definition: y[l] = sum_k w^{(l*k) mod n} x[k]  (Eq. 3) */
static void dft_naive(int n, int sign, const cplx *x, cplx *y)
{
    for (int l = 0; l < n; ++l) {
        cplx acc = 0.0;
        for (int k = 0; k < n; ++k) {
            int64_t e = ((int64_t)l * k) % n;
            acc += orc_root(e, n, sign) * x[k];
        }
        y[l] = acc;
    }
}

/* recursive radix-2 Cooley-Tukey (n = n0 x n1 with n0 = 2):
 * y[k] = E[k] + w_n^k O[k],  y[k + n/2] = E[k] - w_n^k O[k],
 * E = DFT_{n/2}(x even), O = DFT_{n/2}(x odd).  x is read with stride. */
static void dft_radix2(int n, int sign, const cplx *x, int stride, cplx *y, cplx *scratch)
{
    if (n == 1) { y[0] = x[0]; return; }
    int h = n / 2;
    cplx *E = scratch, *O = scratch + h;
    dft_radix2(h, sign, x, 2 * stride, E, scratch + n);
    dft_radix2(h, sign, x + stride, 2 * stride, O, scratch + n);
    for (int k = 0; k < h; ++k) {
        cplx t = orc_root(k, n, sign) * O[k];
        y[k] = E[k] + t;
        y[k + h] = E[k] - t;
    }
}

static int is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

/* one line, contiguous in / out; scratch >= 2 n entries */
static void dft_line(int n, int sign, const cplx *x, cplx *y, cplx *scratch)
{
    if (is_pow2(n)) dft_radix2(n, sign, x, 1, y, scratch);
    else dft_naive(n, sign, x, y);
}

/* exported building blocks, for the pins */
int orc_dft1d(int n, int sign, const cplx *x, cplx *y)
{
    if (n < 1 || (sign != 1 && sign != -1)) return -1;
    cplx *scr = (cplx *)malloc(sizeof(cplx) * 2 * (size_t)n);
    if (!scr) return -2;
    dft_line(n, sign, x, y, scr);
    free(scr);
    return 0;
}

int orc_dft1d_naive(int n, int sign, const cplx *x, cplx *y)
{
    if (n < 1 || (sign != 1 && sign != -1)) return -1;
    dft_naive(n, sign, x, y);
    return 0;
}

/* ------------------------------------------------------------------------ */
/* Cut-off enumeration and the offset array */
/* ------------------------------------------------------------------------ */

/* inclusive ellipsoid test in exact integers:
 *   (k1/a1)^2 + (k2/a2)^2 + (k3/a3)^2 <= 1
 *   <=> k1^2 (a2 a3)^2 + k2^2 (a1 a3)^2 + k3^2 (a1 a2)^2 <= (a1 a2 a3)^2
 * (a_d = 0 means only k_d = 0 on that axis). */
static int in_cutoff(int64_t k1, int64_t k2, int64_t k3, const int32_t a[3])
{
    int64_t a1 = a[0], a2 = a[1], a3 = a[2];
    if ((a1 == 0 && k1 != 0) || (a2 == 0 && k2 != 0) || (a3 == 0 && k3 != 0)) return 0;
    int64_t b1 = a1 ? a1 : 1, b2 = a2 ? a2 : 1, b3 = a3 ? a3 : 1;
    int64_t lhs = k1 * k1 * (b2 * b3) * (b2 * b3) + k2 * k2 * (b1 * b3) * (b1 * b3) +
                  k3 * k3 * (b1 * b2) * (b1 * b2);
    int64_t rhs = (b1 * b2 * b3) * (b1 * b2 * b3);
    return lhs <= rhs;
}

/* Enumerate the cut-off points in packed order: k1 ascending (signed) major,
 * k2 ascending (signed), k3 ascending (signed) fastest (reading R5).
 * Frequencies live in [-N/2, N/2) (R9).  Returns the point count S; fills the
 * arrays when they are non-NULL. */
int64_t orc_enum_points(const int32_t n[3], const int32_t a[3], int32_t *k1, int32_t *k2, int32_t *k3)
{
    int64_t S = 0;
    for (int d = 0; d < 3; ++d)
        if (n[d] < 1 || a[d] < 0 || 2 * a[d] >= n[d]) return -1;
    for (int64_t q1 = -(n[0] / 2); q1 < (n[0] + 1) / 2; ++q1)
        for (int64_t q2 = -(n[1] / 2); q2 < (n[1] + 1) / 2; ++q2)
            for (int64_t q3 = -(n[2] / 2); q3 < (n[2] + 1) / 2; ++q3)
                if (in_cutoff(q1, q2, q3, a)) {
                    if (k1) { k1[S] = (int32_t)q1; k2[S] = (int32_t)q2; k3[S] = (int32_t)q3; }
                    ++S;
                }
    return S;
}

/* The offset array: one entry per non-empty (k1,k2) column ("stick"), in the
 * same order; k3lo = first k3 of the stick, len = its point count,
 * off = exclusive prefix sum of len (n_sticks + 1 entries).  Returns n_sticks,
 * or -3 if a column is not one contiguous k3 range (R6). */
int64_t orc_stick_map(const int32_t n[3], const int32_t a[3], int32_t *sk1, int32_t *sk2, int32_t *k3lo,
                      int32_t *len, int64_t *off)
{
    int64_t S = orc_enum_points(n, a, NULL, NULL, NULL);
    if (S < 0) return -1;
    int32_t *k1 = (int32_t *)malloc(sizeof(int32_t) * 3 * (size_t)(S ? S : 1));
    if (!k1) return -2;
    int32_t *k2 = k1 + S, *k3 = k2 + S;
    orc_enum_points(n, a, k1, k2, k3);
    int64_t ns = 0;
    for (int64_t p = 0; p < S; ++p) {
        int newstick = (p == 0) || k1[p] != k1[p - 1] || k2[p] != k2[p - 1];
        if (newstick) {
            if (sk1) { sk1[ns] = k1[p]; sk2[ns] = k2[p]; k3lo[ns] = k3[p]; len[ns] = 0; off[ns] = p; }
            ++ns;
        } else if (k3[p] != k3[p - 1] + 1) {
            free(k1);
            return -3;
        }
        if (sk1) len[ns - 1] += 1;
    }
    if (sk1) off[ns] = S;
    free(k1);
    return ns;
}

/* ------------------------------------------------------------------------ */
/* Full-cuboid transforms (Eq. 7; 110-112)                   */
/* ------------------------------------------------------------------------ */

static inline int64_t wrap(int64_t k, int64_t n) { int64_t r = k % n; return r < 0 ? r + n : r; }

/* cuboid offset, x fastest (reading R7) */
static inline size_t cub(const int32_t n[3], int64_t i1, int64_t i2, int64_t i3)
{
    return (size_t)i1 + (size_t)n[0] * ((size_t)i2 + (size_t)n[1] * (size_t)i3);
}

/* transform every line of one band's cuboid along `axis` (0 = x, 1 = y, 2 = z) */
static void transform_axis(const int32_t n[3], int axis, int sign, cplx *cube)
{
    int len = n[axis];
    size_t stride = axis == 0 ? 1 : (axis == 1 ? (size_t)n[0] : (size_t)n[0] * n[1]);
    int na = axis == 0 ? n[1] : n[0];             /* the two other extents */
    int nb = axis == 2 ? n[1] : n[2];
    size_t sa = axis == 0 ? (size_t)n[0] : 1;     /* their strides */
    size_t sb = axis == 2 ? (size_t)n[0] : (size_t)n[0] * n[1];
#pragma omp parallel
    {
        cplx *in = (cplx *)malloc(sizeof(cplx) * 4 * (size_t)len);
        cplx *out = in + len, *scr = out + len;
#pragma omp for collapse(2) schedule(static)
        for (int ib = 0; ib < nb; ++ib)
            for (int ia = 0; ia < na; ++ia) {
                cplx *base = cube + ia * sa + ib * sb;
                for (int l = 0; l < len; ++l) in[l] = base[l * stride];
                dft_line(len, sign, in, out, scr);
                for (int l = 0; l < len; ++l) base[l * stride] = out[l];
            }
        free(in);
    }
}

/* inverse: packed sphere -> cuboid.  coef[nb][S], psi[nb][N3][N2][N1].
 * n_axes = 3 for the full transform; 1 = z only, 2 = z then y (stage outputs
 * in the order the paper's staged padding transforms the axes when the stick
 * axis goes first: z, y, x -- any order gives the same final result, Eq. 7). */
int orc_inverse(const int32_t n[3], int64_t S, const int32_t *k1, const int32_t *k2, const int32_t *k3,
                const cplx *coef, cplx *psi, int nb, int n_axes)
{
    if (nb < 1 || n_axes < 0 || n_axes > 3) return -1;
    size_t C = (size_t)n[0] * n[1] * n[2];
    for (int b = 0; b < nb; ++b) {
        cplx *cube = psi + (size_t)b * C;
        memset(cube, 0, sizeof(cplx) * C);
        for (int64_t p = 0; p < S; ++p)
            cube[cub(n, wrap(k1[p], n[0]), wrap(k2[p], n[1]), wrap(k3[p], n[2]))] = coef[(size_t)b * S + p];
        if (n_axes >= 1) transform_axis(n, 2, +1, cube);
        if (n_axes >= 2) transform_axis(n, 1, +1, cube);
        if (n_axes >= 3) transform_axis(n, 0, +1, cube);
    }
    return 0;
}

/* forward: cuboid -> packed sphere, times `scale` (reading R2).  psi is not
 * modified (a private copy of each band is transformed). */
int orc_forward(const int32_t n[3], int64_t S, const int32_t *k1, const int32_t *k2, const int32_t *k3,
                const cplx *psi, cplx *coef, int nb, double scale)
{
    if (nb < 1) return -1;
    size_t C = (size_t)n[0] * n[1] * n[2];
    cplx *cube = (cplx *)malloc(sizeof(cplx) * C);
    if (!cube) return -2;
    for (int b = 0; b < nb; ++b) {
        memcpy(cube, psi + (size_t)b * C, sizeof(cplx) * C);
        transform_axis(n, 0, -1, cube);
        transform_axis(n, 1, -1, cube);
        transform_axis(n, 2, -1, cube);
        for (int64_t p = 0; p < S; ++p)
            coef[(size_t)b * S + p] =
                scale * cube[cub(n, wrap(k1[p], n[0]), wrap(k2[p], n[1]), wrap(k3[p], n[2]))];
    }
    free(cube);
    return 0;
}

/* local-potential apply: c' = forward( V .* inverse(c) ), V real on the grid,
 * shared by all bands (reading R10; PAPER.md:30 motivates the real-space step) */
int orc_apply_vloc(const int32_t n[3], int64_t S, const int32_t *k1, const int32_t *k2, const int32_t *k3,
                   const cplx *coef_in, cplx *coef_out, const double *vloc, int nb, double scale)
{
    if (nb < 1) return -1;
    size_t C = (size_t)n[0] * n[1] * n[2];
    cplx *cube = (cplx *)malloc(sizeof(cplx) * C);
    if (!cube) return -2;
    for (int b = 0; b < nb; ++b) {
        int rc = orc_inverse(n, S, k1, k2, k3, coef_in + (size_t)b * S, cube, 1, 3);
        if (rc) { free(cube); return rc; }
        for (size_t i = 0; i < C; ++i) cube[i] *= vloc[i];
        rc = orc_forward(n, S, k1, k2, k3, cube, coef_out + (size_t)b * S, 1, scale);
        if (rc) { free(cube); return rc; }
    }
    free(cube);
    return 0;
}

/* ------------------------------------------------------------------------ */
/* Brute force: the two defining sums evaluated directly (tiny grids, or a   */
/* handful of sampled outputs on big ones).  Exact integer phase reduction.  */
/* ------------------------------------------------------------------------ */

/* exp(sign j 2 pi (k1 i1/N1 + k2 i2/N2 + k3 i3/N3)), phase reduced exactly
 * over the common denominator L = N1 N2 N3 */
static cplx phase3(const int32_t n[3], int64_t k1, int64_t k2, int64_t k3, int64_t i1, int64_t i2, int64_t i3,
                   int sign)
{
    int64_t L = (int64_t)n[0] * n[1] * n[2];
    int64_t e = (wrap(k1 * i1, n[0]) * ((int64_t)n[1] * n[2]) + wrap(k2 * i2, n[1]) * ((int64_t)n[0] * n[2]) +
                 wrap(k3 * i3, n[2]) * ((int64_t)n[0] * n[1])) % L;
    return orc_root(e, L, sign);
}

/* psi[b][idx] = sum_p c[b][p] exp(+j 2 pi k(p).i/N) for the listed linear
 * cuboid indices idx (Eq. 8).  out[nb][n_idx]. */
int orc_brute_inverse_at(const int32_t n[3], int64_t S, const int32_t *k1, const int32_t *k2, const int32_t *k3,
                         const cplx *coef, int nb, const int64_t *idx, int64_t n_idx, cplx *out)
{
#pragma omp parallel for collapse(2) schedule(static)
    for (int b = 0; b < nb; ++b)
        for (int64_t q = 0; q < n_idx; ++q) {
            int64_t i1 = idx[q] % n[0], i2 = (idx[q] / n[0]) % n[1], i3 = idx[q] / ((int64_t)n[0] * n[1]);
            cplx acc = 0.0;
            for (int64_t p = 0; p < S; ++p)
                acc += coef[(size_t)b * S + p] * phase3(n, k1[p], k2[p], k3[p], i1, i2, i3, +1);
            out[(size_t)b * n_idx + q] = acc;
        }
    return 0;
}

/* c[b][p] = scale * sum_i psi[b][i] exp(-j 2 pi k(p).i/N) for the listed packed
 * indices p (Eq. 3-4).  out[nb][n_idx]. */
int orc_brute_forward_at(const int32_t n[3], const int32_t *k1, const int32_t *k2, const int32_t *k3,
                         const cplx *psi, int nb, const int64_t *pidx, int64_t n_idx, double scale, cplx *out)
{
    size_t C = (size_t)n[0] * n[1] * n[2];
#pragma omp parallel for collapse(2) schedule(static)
    for (int b = 0; b < nb; ++b)
        for (int64_t q = 0; q < n_idx; ++q) {
            int64_t p = pidx[q];
            cplx acc = 0.0;
            for (int64_t i3 = 0; i3 < n[2]; ++i3)
                for (int64_t i2 = 0; i2 < n[1]; ++i2)
                    for (int64_t i1 = 0; i1 < n[0]; ++i1)
                        acc += psi[(size_t)b * C + cub(n, i1, i2, i3)] *
                               phase3(n, k1[p], k2[p], k3[p], i1, i2, i3, -1);
            out[(size_t)b * n_idx + q] = scale * acc;
        }
    return 0;
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
