// fftb_plane_fast.cuh -- warp-synchronous building blocks and z-pass kernels for half-band power-of-two
// grids (sm_100a); the plane kernel built from them is in fftb_plane_pf.cuh.
//
// Same mathematics as plane_k in fftb_kernels.cuh (y and x passes of one z-plane, one y residue per
// CTA; PAPER.md:96 Fig. 3, :112 staged padding), restructured for the B200 SM:
//   * a length-N half-band line is two length-M = N/2 transforms (n = 2n' + e) of
//         u_e[k_s mod M] = x[k_s] W^{e k_s},   k_s the SIGNED frequency in [-M/2, M/2], W = exp(+2 pi j/N)
//     (the two aliases k_s = -M/2, +M/2 share slot M/2).  No index shift and no output modulation;
//     the e = 0 half has no arithmetic in front of it at all: that is the pruning of the first stage.
//   * a length-M transform is done by a GROUP of P2 lanes of one warp, P1 = M/P2 values per lane,
//     two in-register codelet stages around one exchange through a warp-private shared-memory
//     tile: only __syncwarp, no CTA barrier inside a transform.
//   * the inter-stage twiddles W^{2 t m} (t = lane in group) live in registers for the whole kernel;
//     the e = 1 pre-twiddle is W^t (one register pair) times a compile-time root of order 2 P1.
//   * the forward direction is the exact adjoint chain, so in VLOC mode the line never leaves the
//     registers between the inverse x pass, the V(r) multiply and the forward x pass.
//   * the only CTA-wide barriers are the two between the y and x passes (plane buffer hand-over).
#pragma once
#include "fftb_kernels.cuh"

namespace fftb {

template <typename T, int N_, int P1_, int P2_> struct FastCfg {
    static constexpr int N = N_, P1 = P1_, P2 = P2_, M = N_ / 2;
    static constexpr int G = 32 / P2_;   // transforms per warp
    static constexpr int B2 = P1_ / P2_; // stage-2 codelets per lane
    static constexpr int LW = 128 / (int)sizeof(cx<T>); // lanes per shared-memory wavefront
    // plane buffer pitch: >= M, congruent to LW/P2 modulo LW (conflict-free column-strided reads)
    static constexpr int YP = M + ((LW / P2_ - M % LW) + LW) % LW;
    static constexpr int NCOL = M + 1;
    static constexpr int FS0 = P1_ * (P2_ + 1);
    static constexpr int FS = P2_ >= 8 ? FS0 : FS0 + ((P2_ - FS0 % 8) + 8) % 8; // tile pitch per transform
    static constexpr int EXW = G * FS;   // exchange elements per warp
    static_assert(P1_ * P2_ * 2 == N_ && P1_ % P2_ == 0 && 32 % P2_ == 0 && 96 % (2 * P1_) == 0, "unsupported factorisation");
    static constexpr size_t smem_bytes(int nwarps) { return sizeof(cx<T>) * ((size_t)NCOL * YP + (size_t)nwarps * EXW); }
};

// Column table of the y pass, passed BY VALUE as a kernel parameter (constant bank): no dependent
// global loads stand between the start of a CTA and its first loads of the intermediate A.
constexpr int FAST_MAXCOL = 65; // N <= 128: at most N/2 + 1 occupied k1 columns
struct ColTab {
    int4 col[FAST_MAXCOL];  // {first stick, stick count, k2lo, 0} per occupied k1 column
    int perm[FAST_MAXCOL];  // multi-stick columns first, then the single-stick ones
};

// Column (index into the plan's column permutation) of lane group f in y task `task`, and the number of y tasks.
// A shared-memory wavefront covers GW = LW / P2 lane groups x P2 consecutive elements of their columns.  The
// plane-buffer pitch is congruent to GW modulo LW (what the x pass needs), so the GW columns of one wavefront
// must be D = P2 / GW columns apart to fall into different banks: the y tasks take their columns from blocks of
// GW x D columns, wavefront r of a block the columns r, r + D, ...  (identity when GW = 1 or D = 1).
template <class F> __device__ __forceinline__ int ycol_index(int task, int f)
{
    constexpr int GW = F::LW / F::P2 < 1 ? 1 : F::LW / F::P2, D = F::P2 / GW;
    if constexpr (GW <= 1 || D <= 1) {
        return task * F::G + f;
    } else {
        static_assert(F::G % GW == 0, "lane groups per warp must be a multiple of the groups per wavefront");
        const int u = f % GW, w = task * (F::G / GW) + f / GW;
        return (w / D) * (GW * D) + u * D + (w % D);
    }
}
template <class F> __host__ __device__ __forceinline__ int ycol_tasks(int n_multi)
{
    constexpr int GW = F::LW / F::P2 < 1 ? 1 : F::LW / F::P2, D = F::P2 / GW;
    constexpr int BLK = (GW <= 1 || D <= 1) ? 1 : GW * D;
    return ((n_multi + BLK - 1) / BLK * BLK + F::G - 1) / F::G;
}

// signed frequency held by lane t in slot j (slot P1/2 of lane 0 is the -M/2 alias; +M/2 is extra)
template <class F> __device__ __forceinline__ int ks_of(int t, int j) { return t + F::P2 * j - (j >= F::P1 / 2 ? F::M : 0); }
// order-2P1 root index of the e = 1 pre-twiddle of slot j (the sign of the wrapped half is folded in)
template <class F> __host__ __device__ constexpr int jroot(int j) { return j < F::P1 / 2 ? j : j + F::P1; }

// e = 1 pre-twiddle (inverse): x[j] *= W^t * w_{2P1}^{jroot(j)}
template <class F, int J, typename T> __device__ __forceinline__ void pre_inv(cx<T> (&x)[F::P1], cx<T> g)
{
    if constexpr (J < F::P1) {
        x[J] = mul_root<jroot<F>(J), 2 * F::P1, +1, T>(cmul(x[J], g));
        pre_inv<F, J + 1, T>(x, g);
    }
}
// forward combine: F[j] = G0[j] + conj(W^t w^{jroot(j)}) G1[j]; returns the G1 term in g1
template <class F, int J, typename T> __device__ __forceinline__ void post_fwd(cx<T> (&g1)[F::P1], cx<T> g)
{
    if constexpr (J < F::P1) {
        g1[J] = cmulc(mul_root<jroot<F>(J), 2 * F::P1, -1, T>(g1[J]), g);
        post_fwd<F, J + 1, T>(g1, g);
    }
}

// conj twiddle w_{P1}^{t' b} of the forward first stage for codelet b > 0
template <class F, int B, int TP, typename T> __device__ __forceinline__ void fwd_btw(cx<T> (&y)[F::P2])
{
    if constexpr (TP < F::P2) {
        y[TP] = mul_root<TP * B, F::P1, -1, T>(y[TP]);
        fwd_btw<F, B, TP + 1, T>(y);
    }
}
template <class F, int B, typename T> __device__ __forceinline__ void fwd_btw_all(cx<T> (&y)[F::B2][F::P2])
{
    if constexpr (B < F::B2) {
        if constexpr (B > 0) fwd_btw<F, B, 1, T>(y[B]);
        fwd_btw_all<F, B + 1, T>(y);
    }
}

// Where a group exchanges its M values between the two codelet stages: element (i, j), i < P1 the
// stage-1 output index, j < P2 the lane.  ExTile is a warp-private tile of pitch P2+1; ExSkew uses M
// slots that lie STRIDE elements apart (a line or a column of the plane buffer, exchanged in place),
// rotated by i so that both access directions touch P2 different 16-byte bank groups.
template <typename T, int P2> struct ExTile {
    cx<T> *p;
    __device__ __forceinline__ void put(int i, int j, cx<T> v) const { p[i * (P2 + 1) + j] = v; }
    __device__ __forceinline__ cx<T> get(int i, int j) const { return p[i * (P2 + 1) + j]; }
};
template <typename T, int P2, int STRIDE> struct ExSkew {
    cx<T> *p;
    bool on; // a group without work must not scribble over somebody else's line or column
    __device__ __forceinline__ int slot(int i, int j) const { return (P2 * i + ((j + i) & (P2 - 1))) * STRIDE; }
    __device__ __forceinline__ void put(int i, int j, cx<T> v) const { if (on) p[slot(i, j)] = v; }
    __device__ __forceinline__ cx<T> get(int i, int j) const { return p[slot(i, j)]; }
};

// length-M inverse transform of the group: x[j] = u[t + P2 j]  ->  y[b][q] = out[(t + P2 b) + P1 q]
template <class F, typename T, class EX>
__device__ __forceinline__ void sub_inv(cx<T> (&x)[F::P1], cx<T> (&y)[F::B2][F::P2], const cx<T> (&tws)[F::P1], EX ex, int t)
{
    constexpr int P1 = F::P1, P2 = F::P2, B2 = F::B2;
    fft_reg<P1, +1, T>(x);
#pragma unroll
    for (int m = 1; m < P1; ++m) x[m] = cmul(x[m], tws[m]);
    __syncwarp();
#pragma unroll
    for (int m = 0; m < P1; ++m) ex.put(m, t, x[m]);
    __syncwarp();
#pragma unroll
    for (int b = 0; b < B2; ++b) {
#pragma unroll
        for (int tt = 0; tt < P2; ++tt) y[b][tt] = ex.get(t + P2 * b, tt);
        fft_reg<P2, +1, T>(y[b]);
    }
}

// adjoint: y[b][q] = in[(t + P2 b) + P1 q]  ->  x[j] = G[t + P2 j]
template <class F, typename T, class EX>
__device__ __forceinline__ void sub_fwd(cx<T> (&y)[F::B2][F::P2], cx<T> (&x)[F::P1], const cx<T> (&tws)[F::P1], EX ex, int t)
{
    constexpr int P1 = F::P1, P2 = F::P2, B2 = F::B2;
#pragma unroll
    for (int b = 0; b < B2; ++b) {
        fft_reg<P2, -1, T>(y[b]);
#pragma unroll
        for (int tt = 1; tt < P2; ++tt) y[b][tt] = cmulc(y[b][tt], tws[tt]);
    }
    fwd_btw_all<F, 0, T>(y);
    __syncwarp();
#pragma unroll
    for (int b = 0; b < B2; ++b)
#pragma unroll
        for (int tt = 0; tt < P2; ++tt) ex.put(t + P2 * b, tt, y[b][tt]);
    __syncwarp();
#pragma unroll
    for (int m = 0; m < P1; ++m) x[m] = ex.get(m, t);
    fft_reg<P1, -1, T>(x);
}

// The two halves of sub_inv / sub_fwd: everything in front of the exchange works on registers only, so a warp may do it
// before it is allowed to touch the shared-memory line or column the exchange happens in (split barriers of plane_pf_k).
// front + back = the same arithmetic in the same order as the whole.
template <class F, typename T>
__device__ __forceinline__ void sub_inv_front(cx<T> (&x)[F::P1], const cx<T> (&tws)[F::P1])
{
    fft_reg<F::P1, +1, T>(x);
#pragma unroll
    for (int m = 1; m < F::P1; ++m) x[m] = cmul(x[m], tws[m]);
}
template <class F, typename T, class EX>
__device__ __forceinline__ void sub_inv_back(cx<T> (&x)[F::P1], cx<T> (&y)[F::B2][F::P2], EX ex, int t)
{
    constexpr int P1 = F::P1, P2 = F::P2, B2 = F::B2;
    __syncwarp();
#pragma unroll
    for (int m = 0; m < P1; ++m) ex.put(m, t, x[m]);
    __syncwarp();
#pragma unroll
    for (int b = 0; b < B2; ++b) {
#pragma unroll
        for (int tt = 0; tt < P2; ++tt) y[b][tt] = ex.get(t + P2 * b, tt);
        fft_reg<P2, +1, T>(y[b]);
    }
}
template <class F, typename T>
__device__ __forceinline__ void sub_fwd_front(cx<T> (&y)[F::B2][F::P2], const cx<T> (&tws)[F::P1])
{
#pragma unroll
    for (int b = 0; b < F::B2; ++b) {
        fft_reg<F::P2, -1, T>(y[b]);
#pragma unroll
        for (int tt = 1; tt < F::P2; ++tt) y[b][tt] = cmulc(y[b][tt], tws[tt]);
    }
    fwd_btw_all<F, 0, T>(y);
}
template <class F, typename T, class EX>
__device__ __forceinline__ void sub_fwd_back(cx<T> (&y)[F::B2][F::P2], cx<T> (&x)[F::P1], EX ex, int t)
{
    constexpr int P1 = F::P1, P2 = F::P2, B2 = F::B2;
    __syncwarp();
#pragma unroll
    for (int b = 0; b < B2; ++b)
#pragma unroll
        for (int tt = 0; tt < P2; ++tt) ex.put(t + P2 * b, tt, y[b][tt]);
    __syncwarp();
#pragma unroll
    for (int m = 0; m < P1; ++m) x[m] = ex.get(m, t);
    fft_reg<P1, -1, T>(x);
}

// ---------------------------------------------------------------------------------------------
// z passes, warp-synchronous: one group of P2 lanes per stick, G sticks per warp, TS = G * NW
// consecutive sticks per CTA.  The transposition between "one stick, all z" (what a transform
// produces / consumes) and the plane-major intermediate A[z][stick] goes through a shared-memory
// tile [N][TS] so that every global access to A is a run of TS consecutive elements of one z row
// (512 bytes for complex128); element (z, sl) sits in column (sl + z/2) mod TS, which makes the
// strided accesses of the transforms bank-conflict-free.
//   grid = (ceil(n_sticks / TS), bands)
// ---------------------------------------------------------------------------------------------
template <typename T, class F, int NW> struct ZFast {
    static constexpr int TS = F::G * NW;
    // a shared-memory wavefront covers GW = LW / P2 lane groups (sticks) x P2 lanes (rows z, z+2, ...): the row
    // rotation steps by GW so that those LW accesses fall into different banks in either precision
    static constexpr int GW = F::LW / F::P2 < 1 ? 1 : F::LW / F::P2;
    static_assert(TS >= F::LW, "tile row shorter than a wavefront");
    __device__ static __forceinline__ int rot(int z) { return (z >> 1) * GW; }
    __device__ static __forceinline__ int swz(int z, int sl) { return z * TS + ((sl + rot(z)) & (TS - 1)); }
    // tile of the persistent kernels (fftb_zpass_pf.cuh; rows move by TMA bulk copies, so every row must be one
    // contiguous, 16-byte aligned run):
    // the rows z = 2m, 2m + 1 form a pair of pitch RP = 2 TS + GW elements; the P2 lanes of a group write the
    // rows z, z + 2, ... of one column, GW groups per wavefront the neighbouring columns: (m RP + sl) mod LW
    // takes LW different values
    static constexpr int RP = 2 * TS + GW;
    static_assert((RP * sizeof(cx<T>)) % 16 == 0 && (TS * sizeof(cx<T>)) % 16 == 0, "bulk copies need 16-byte aligned rows");
    __device__ static __forceinline__ int lin(int z, int sl) { return (z >> 1) * RP + (z & 1) * TS + sl; }
    static constexpr int TILE = (F::N / 2) * RP; // >= N TS: both layouts fit
    static constexpr size_t smem_bytes = sizeof(cx<T>) * ((size_t)TILE + (size_t)NW * F::EXW);
};

// TMA bulk store shared -> global (bulk async-group completion)
__device__ __forceinline__ void bulk_store(void *gdst, const void *ssrc, unsigned bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst),
                 "r"((unsigned)__cvta_generic_to_shared(ssrc)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void bulk_store_commit_wait_read()
{
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}

// One tile (TS consecutive sticks starting at s0 = j TS) of one band, called by all NW warps of a CTA;
// `smem` holds the tile [N][TS] and the warps' exchange tiles (ZFast::smem_bytes); tws / g are the caller's
// twiddle registers for the z axis.  Contains CTA barriers.  Forward only: the inverse z pass and the forward one
// with a single plane of A are the persistent kernels of fftb_zpass_pf.cuh.
template <typename T, class F, int NW>
__device__ __forceinline__ void z_fwd_tile(const DevPlan &pl, const cx<T> *__restrict__ A_band, cx<T> *__restrict__ packed_band, int j,
                                           cx<T> *smem, const cx<T> (&tws)[F::P1], cx<T> g)
{
    using C = cx<T>;
    using Z = ZFast<T, F, NW>;
    constexpr int N = F::N, M = F::M, P1 = F::P1, P2 = F::P2, B2 = F::B2, G = F::G, TS = Z::TS, NT = NW * 32;
    C *tile = smem;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int f = lane / P2, t = lane % P2;
    const ExTile<T, P2> ex{tile + Z::TILE + warp * F::EXW + f * F::FS};
    const int s0 = j * TS, sl = warp * G + f, s = s0 + sl;
    const bool act = s < pl.nsticks;
    // ---- A[z][s0 .. s0+TS) -> tile, summing the ry partial planes of the generic forward plane kernel
    {
        const C *src = A_band + s0;
        const long long rstride = (long long)pl.n3 * pl.pitch;
        constexpr int U = 8;
        static_assert((N * TS) % (NT * U) == 0, "tile copy is unrolled by U");
        for (int i0 = tid; i0 < N * TS; i0 += NT * U) {
            C v[U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int i = i0 + u * NT, z = i / TS, l = i % TS;
                v[u] = (s0 + l < pl.nsticks) ? __ldcg(src + (long long)z * pl.pitch + l) : czero<T>();
            }
            for (int p = 1; p < pl.ry; ++p) {
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    const int i = i0 + u * NT, z = i / TS, l = i % TS;
                    if (s0 + l < pl.nsticks) v[u] = cadd(v[u], __ldcg(src + p * rstride + (long long)z * pl.pitch + l));
                }
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int i = i0 + u * NT, z = i / TS, l = i % TS;
                tile[Z::swz(z, l)] = v[u];
            }
        }
    }
    const int4 st = pl.stick[act ? s : 0];
    C *dst = packed_band + st.x;
    const T scale = (T)pl.scale;
    __syncthreads();
    C y[B2][P2], g0[P1], g1[P1];
#pragma unroll
    for (int bb = 0; bb < B2; ++bb)
#pragma unroll
        for (int q = 0; q < P2; ++q) y[bb][q] = tile[Z::swz(2 * ((t + P2 * bb) + P1 * q), sl)];
    sub_fwd<F, T>(y, g0, tws, ex, t);
#pragma unroll
    for (int bb = 0; bb < B2; ++bb)
#pragma unroll
        for (int q = 0; q < P2; ++q) y[bb][q] = tile[Z::swz(2 * ((t + P2 * bb) + P1 * q) + 1, sl)];
    sub_fwd<F, T>(y, g1, tws, ex, t);
    post_fwd<F, 0, T>(g1, g);
    if (act) {
        const int idb = M / 2 - st.y;
        if (t == 0 && (unsigned)idb < (unsigned)st.z) {
            const C v = csub(g0[P1 / 2], g1[P1 / 2]);
            dst[idb] = mk<T>(v.x * scale, v.y * scale);
        }
#pragma unroll
        for (int jj = 0; jj < P1; ++jj) {
            const int idx = ks_of<F>(t, jj) - st.y;
            if ((unsigned)idx < (unsigned)st.z) {
                const C v = cadd(g0[jj], g1[jj]);
                dst[idx] = mk<T>(v.x * scale, v.y * scale);
            }
        }
    }
}

// stand-alone forward z-pass kernel: one tile per CTA, grid = (ceil(n_sticks / TS), bands)
template <typename T, class F, int NW>
__global__ void __launch_bounds__(NW * 32, F::P1 > 16 ? 2 : 16 / NW)
zpass_fast_fwd_k(const __grid_constant__ DevPlan pl, const cx<T> *__restrict__ A, cx<T> *__restrict__ packed, long long a_band_stride)
{
    using C = cx<T>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int t = (threadIdx.x & 31) % F::P2;
    const C *tw = reinterpret_cast<const C *>(pl.tw3);
    C tws[F::P1];
#pragma unroll
    for (int m = 1; m < F::P1; ++m) tws[m] = tw[modn<F::N>(2 * t * m)];
    tws[0] = mk<T>((T)1, (T)0);
    z_fwd_tile<T, F, NW>(pl, A + (long long)blockIdx.y * a_band_stride, packed + (long long)blockIdx.y * pl.S, blockIdx.x,
                         reinterpret_cast<C *>(smem_raw), tws, tw[t]);
}

} // namespace fftb
