// fftb_dense.cuh -- the dense (unpruned) comparison arm on the warp-synchronous transform core (sm_100a).
//
// "zero-pad the entire sphere ... the 3D Fourier computation is applied on the entire cube" -- the
// route FFTB's staged padding is measured against (BASELINE config 5).  Nothing can be pruned here: every (k1,k2) is a
// full-length stick, every line of every pass carries data on the whole band, so the transform is three plain passes
// over the cube per direction.  ONE kernel does all of them: G = 32 / P2 lines per warp, one lane group per line, the
// line held in registers, both halves of the first radix-2 split carrying data:
//       u_0[k mod M] = x[k_a] + x[k_b],  u_1[k mod M] = (x[k_a] - x[k_b]) W^{k_a},   k_a in [-M/2, M/2), k_b = k_a -/+ M
// (W^{+-M} = -1), then the two length-M transforms of fftb_plane_fast.cuh (sub_inv / sub_fwd, n = 2n' + e); the
// forward direction is the adjoint chain.  A pass is described by element strides (DenseGeom), which is also how the
// transposition between the packed order [k1][k2][k3] and the cuboid [z][y][x] happens: the z pass writes the
// plane-major intermediate A[z][k1][k2] the pruned kernels use (pitch N1 N2), the y pass works on A in place, the x
// pass reads A with stride N2 and writes cuboid rows (the mirror image forward).  Lines that are neighbours in
// memory sit in neighbouring lane groups and warps, so a strided access still fills whole 32-byte sectors
// (G x 16 bytes for complex128); there is no shared-memory staging, the 126 MB L2 merges the sectors of a row.
#pragma once
#include "fftb_plane_fast.cuh"

namespace fftb {

struct DenseGeom {
    long long in_u, in_v, in_i;    // element strides of the input: slow line index u, fast line index v, position on the line
    long long out_u, out_v, out_i; // the same for the output
    long long in_band, out_band;   // elements per band
    int nv;                        // line L = u * nv + v
    int lines;                     // lines per band
};

enum DenseMode { DENSE_INV = 0, DENSE_FWD = 1, DENSE_VLOC = 2 };

// position of signed frequency k on a frequency-ordered line (packed dense order: k + N/2)
template <class F> __device__ __forceinline__ int dense_pos(int k) { return k + F::M; }

// MODE INV:  in frequency-ordered, out natural (n = 0..N-1);  FWD: in natural, out frequency-ordered, times `scale`;
// VLOC (x axis only): in and out frequency-ordered, the natural-order line is multiplied by vloc[line][n] in between.
// PAIR: the natural-order side is contiguous (stride 1): its (2n', 2n'+1) pairs move as one access.
template <typename T, class F, int NW, int MODE, bool PAIR>
__global__ void __launch_bounds__(NW * 32)
dense_axis_k(const cx<T> *__restrict__ in, cx<T> *__restrict__ out, const __grid_constant__ DenseGeom ge, const cx<T> *__restrict__ tw,
             const T *__restrict__ vloc, T scale)
{
    using C = cx<T>;
    constexpr int N = F::N, M = F::M, P1 = F::P1, P2 = F::P2, B2 = F::B2, G = F::G;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int f = lane / P2, t = lane % P2;
    const ExTile<T, P2> ex{reinterpret_cast<C *>(smem_raw) + warp * F::EXW + f * F::FS};
    C tws[P1];
#pragma unroll
    for (int m = 1; m < P1; ++m) tws[m] = tw[modn<N>(2 * t * m)];
    tws[0] = mk<T>((T)1, (T)0);
    const C g = tw[t];
    const int L = (blockIdx.x * NW + warp) * G + f;
    const bool act = L < ge.lines;
    const int u = act ? L / ge.nv : 0, v = act ? L % ge.nv : 0;
    const C *src = in + (long long)blockIdx.y * ge.in_band + u * ge.in_u + v * ge.in_v;
    C *dst = out + (long long)blockIdx.y * ge.out_band + u * ge.out_u + v * ge.out_v;
    C y0[B2][P2], y1[B2][P2];
    if constexpr (MODE != DENSE_FWD) {
        C s[P1], d[P1];
#pragma unroll
        for (int j = 0; j < P1; ++j) {
            const int ka = ks_of<F>(t, j), kb = ka < 0 ? ka + M : ka - M;
            const C xa = act ? __ldcs(src + dense_pos<F>(ka) * ge.in_i) : czero<T>();
            const C xb = act ? __ldcs(src + dense_pos<F>(kb) * ge.in_i) : czero<T>();
            s[j] = cadd(xa, xb);
            d[j] = csub(xa, xb);
        }
        sub_inv<F, T>(s, y0, tws, ex, t);
        pre_inv<F, 0, T>(d, g);
        sub_inv<F, T>(d, y1, tws, ex, t);
    }
    if constexpr (MODE == DENSE_INV) {
        if (act) {
#pragma unroll
            for (int bb = 0; bb < B2; ++bb)
#pragma unroll
                for (int q = 0; q < P2; ++q) {
                    const int np = (t + P2 * bb) + P1 * q;
                    if constexpr (PAIR) st_pair(dst + 2 * np, y0[bb][q], y1[bb][q]);
                    else {
                        __stcs(dst + (2 * np) * ge.out_i, y0[bb][q]);
                        __stcs(dst + (2 * np + 1) * ge.out_i, y1[bb][q]);
                    }
                }
        }
        return;
    }
    if constexpr (MODE == DENSE_VLOC) {
        const T *vrow = vloc + (long long)L * N; // the x axis: line L = z N2 + y of V[z][y][x]
#pragma unroll
        for (int bb = 0; bb < B2; ++bb)
#pragma unroll
            for (int q = 0; q < P2; ++q) {
                const int np = (t + P2 * bb) + P1 * q;
                const T v0 = act ? vrow[2 * np] : (T)0, v1 = act ? vrow[2 * np + 1] : (T)0;
                y0[bb][q].x *= v0; y0[bb][q].y *= v0;
                y1[bb][q].x *= v1; y1[bb][q].y *= v1;
            }
    }
    if constexpr (MODE == DENSE_FWD) {
#pragma unroll
        for (int bb = 0; bb < B2; ++bb)
#pragma unroll
            for (int q = 0; q < P2; ++q) {
                const int np = (t + P2 * bb) + P1 * q;
                if (!act) { y0[bb][q] = czero<T>(); y1[bb][q] = czero<T>(); }
                else if constexpr (PAIR) ld_pair(src + 2 * np, y0[bb][q], y1[bb][q]);
                else {
                    y0[bb][q] = __ldcs(src + (2 * np) * ge.in_i);
                    y1[bb][q] = __ldcs(src + (2 * np + 1) * ge.in_i);
                }
            }
    }
    C g0[P1], g1[P1];
    sub_fwd<F, T>(y0, g0, tws, ex, t);
    sub_fwd<F, T>(y1, g1, tws, ex, t);
    post_fwd<F, 0, T>(g1, g);
    if (act) {
#pragma unroll
        for (int j = 0; j < P1; ++j) {
            const int ka = ks_of<F>(t, j), kb = ka < 0 ? ka + M : ka - M;
            const C a = cadd(g0[j], g1[j]), b = csub(g0[j], g1[j]);
            __stcs(dst + dense_pos<F>(ka) * ge.out_i, mk<T>(a.x * scale, a.y * scale));
            __stcs(dst + dense_pos<F>(kb) * ge.out_i, mk<T>(b.x * scale, b.y * scale));
        }
    }
}

} // namespace fftb
