// fftb_plane_pf.cuh -- persistent plane kernel with register prefetch (sm_100a).
//
// Same mathematics and the same building blocks as fftb_plane_fast.cuh (half-band line = two length-M
// transforms done by groups of P2 lanes around one warp-private exchange tile; Fig. 3,
// :112 staged padding).  What this kernel changes is the schedule:
//   * measured on B200 (profiles/): the transform core alone (register
//     butterflies + the shared-memory exchange) already runs at the FP64 pipe's rate with 8 warps per
//     SM; what held the plane kernel at 45% of every pipe was that each iteration waited, in every
//     warp at the same time, for global memory (the stick values of the plane, the cuboid lines).
//   * so a CTA has only NW = (x tasks per half plane)/2 warps, each with up to 255 registers, and
//     every global load is issued ONE TASK AHEAD into registers: the y-pass input of task it+1 while
//     the x pass of task it-1 runs, the cuboid lines (and V(r)) of the next x task while the current
//     one is transformed.  No warp ever waits for DRAM or L2 with nothing else in flight.
//
// A TASK is one half z-plane (band b, plane z, y residue r), id = (b * n3 + z) * 2 + r; CTA c of a
// persistent grid of G CTAs owns tasks c, c + G, ...  The plane buffer is double-buffered:
//   INV   it: y_inv(task it) -> buf[it&1]                | x_inv(task it-1): buf[(it-1)&1] -> cuboid
//   FWD   it: x_fwd(task it) -> buf[it&1]                | y_fwd(task it-1): buf[(it-1)&1] -> A
//   VLOC  it: y_fwd(task it-2): buf[it&1] -> A, then y_inv(task it) -> buf[it&1] (same warp, same
//             columns, in this order)                    | x_vloc(task it-1) in place in buf[(it-1)&1]
// with one CTA-wide barrier per iteration.
#pragma once
#include "fftb_plane_fast.cuh"

namespace fftb {

template <typename T, class F, int NW> struct PlanePF {
    static constexpr int PB = F::NCOL * F::YP;       // elements of one plane buffer
    static constexpr int NXT = F::M / F::G;          // x tasks per half plane (G lines each)
    static constexpr int XT = NXT / NW;              // x tasks per warp and iteration
    static constexpr int YT = 2;                     // y tasks per warp whose input is prefetched
    static_assert(NXT % NW == 0 && XT >= 1, "x tasks must divide evenly over the warps");
    static constexpr size_t smem_bytes = sizeof(cx<T>) * (2 * (size_t)PB + (size_t)NW * F::EXW);
    // INV, VLOC: plane buffers, exchange tiles, one staged row of A (pitch elements).
    // FWD: plane buffers (the exchanges are done in place in them), G staged cuboid lines per warp.
    static size_t smem_bytes_mode(int mode, int pitch)
    {
        if (mode == MODE_FWD) return sizeof(cx<T>) * (2 * (size_t)PB + (size_t)NW * F::G * F::N);
        return smem_bytes + sizeof(cx<T>) * (size_t)pitch;
    }
};

struct PlaneTask { int b, z, r; };

// ---- mbarrier + TMA bulk copy (global -> shared), the asynchronous path that does not occupy a
// scoreboard slot while it is in flight (register prefetch across a whole x pass does, and every
// later wait on that slot then waits for the prefetch too) --------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity)
{
    unsigned done;
    do {
        asm volatile("{\n\t.reg .pred p;\n\t"
                     "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                     "selp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done)
                     : "r"(smem_u32(bar)), "r"(parity)
                     : "memory");
    } while (!done);
}
__device__ __forceinline__ void bulk_load(void *sdst, const void *gsrc, unsigned bytes, unsigned long long *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(sdst)),
                 "l"(gsrc), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

template <typename T, class F, int NW, int MODE>
__global__ void __launch_bounds__(NW * 32, 1)
plane_pf_k(const __grid_constant__ DevPlan pl, const __grid_constant__ ColTab ct, const cx<T> *__restrict__ Ain,
           cx<T> *__restrict__ Aout, const cx<T> *__restrict__ cub_in, cx<T> *__restrict__ cub_out,
           const T *__restrict__ vloc, long long a_in_stride, long long a_out_stride, int ntasks)
{
    using C = cx<T>;
    using PF = PlanePF<T, F, NW>;
    constexpr int N = F::N, M = F::M, P1 = F::P1, P2 = F::P2, B2 = F::B2, G = F::G, YP = F::YP;
    constexpr int PB = PF::PB, XT = PF::XT, YT = PF::YT;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C *pbuf0 = reinterpret_cast<C *>(smem_raw); // [2][NCOL][YP]: column c = k1 - k1lo, local line y'
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int f = lane / P2, t = lane % P2;
    const ExTile<T, P2> ex{pbuf0 + 2 * PB + warp * F::EXW + f * F::FS}; // this group's exchange tile
    // INV, VLOC: landing zone of the next plane's row A[b][z][0..pitch) (one TMA bulk copy per task)
    C *stage = pbuf0 + 2 * PB + NW * F::EXW;
    __shared__ __align__(8) unsigned long long bar_full, bar_empty, bar_line[NW];
    // FWD: landing zone of this warp's next x task, G cuboid lines (no tiles in this mode)
    C *lstage = pbuf0 + 2 * PB + warp * (G * N);
    unsigned line_par = 0;
    const unsigned stage_bytes = (unsigned)pl.pitch * (unsigned)sizeof(C);
    const C *tw = reinterpret_cast<const C *>(pl.tw1);  // N1 == N2: one table
    C tws[P1];
#pragma unroll
    for (int m = 1; m < P1; ++m) tws[m] = tw[modn<N>(2 * t * m)];
    tws[0] = mk<T>((T)1, (T)0);
    const C g = tw[t];
    const int nx = pl.nxocc, k1lo = pl.k1lo;
    const bool l0 = (t == 0);
    const int n_one = nx - pl.n_multi;
    const int ntask_y = (pl.n_multi + G - 1) / G;
    const int ktasks = ntasks > (int)blockIdx.x ? (ntasks - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;
    constexpr int LAG = (MODE == MODE_VLOC) ? 2 : 1; // iterations between the first and the last stage of a task

    auto decode = [&](int k) -> PlaneTask {
        const int id = blockIdx.x + k * gridDim.x;
        PlaneTask q;
        q.r = id & 1;
        q.z = (id >> 1) % pl.n3;
        q.b = (id >> 1) / pl.n3;
        return q;
    };
    // column group of this lane in y task `task`; those of the warp's first YT tasks never change
    struct YCol { bool act; int col; int4 co; };
    auto ycol = [&](int task) -> YCol {
        YCol c;
        const int ci = task * G + f;
        c.act = task < ntask_y && ci < pl.n_multi;
        c.col = ct.perm[c.act ? ci : 0];
        c.co = ct.col[c.col];
        return c;
    };
    YCol yc[YT];
#pragma unroll
    for (int u = 0; u < YT; ++u) yc[u] = ycol(warp + u * NW);
    // single-stick column of this warp (closed form), if any
    const bool one_act = warp < n_one;
    const int one_col = ct.perm[pl.n_multi + (one_act ? warp : 0)];
    const int4 one_co = ct.col[one_col];

    // ---- loads that run one task ahead -----------------------------------------------------------
    // stick values of one column group (inverse y pass input) from the staged row of A
    auto yinv_load = [&](const YCol &c, C (&x)[P1], C &bv) {
        const C *src = stage + c.co.x;
#pragma unroll
        for (int j = 0; j < P1; ++j) {
            const int idx = ks_of<F>(t, j) - c.co.z;
            x[j] = (c.act && (unsigned)idx < (unsigned)c.co.y) ? src[idx] : czero<T>();
        }
        const int idb = M / 2 - c.co.z;
        bv = (c.act && l0 && (unsigned)idb < (unsigned)c.co.y) ? src[idb] : czero<T>();
    };
    // one thread asks the TMA engine for the row of task tk; completion is signalled on bar_full
    auto stage_issue = [&](const PlaneTask &tk) {
        mbar_expect_tx(&bar_full, stage_bytes);
        bulk_load(stage, Ain + (long long)tk.b * a_in_stride + (long long)tk.z * pl.pitch, stage_bytes, &bar_full);
    };
    // FWD: the G cuboid lines of x task u are fetched by the TMA engine into this warp's landing zone
    auto line_issue = [&](const PlaneTask &tk, int u) {
        if (lane == 0) mbar_expect_tx(&bar_line[warp], (unsigned)(G * N * sizeof(C)));
        __syncwarp();
        if (lane < G) {
            const int yl = (warp + u * NW) * G + lane;
            bulk_load(lstage + lane * N, cub_in + (((long long)tk.b * pl.n3 + tk.z) * N + (2 * yl + tk.r)) * N,
                      (unsigned)(N * sizeof(C)), &bar_line[warp]);
        }
    };
    // ... and read from there as (x, x+1) pairs; half of the lanes take the odd element first so that
    // the 32-byte-strided 16-byte reads of a quarter warp fall into different bank groups
    auto line_read = [&](C (&o0)[B2][P2], C (&o1)[B2][P2]) {
        mbar_wait(&bar_line[warp], line_par);
        line_par ^= 1u;
        const bool sw = (P2 >= 8) ? (t >= P2 / 2) : ((f & 1) != 0);
        const C *st = lstage + f * N;
#pragma unroll
        for (int bb = 0; bb < B2; ++bb)
#pragma unroll
            for (int q = 0; q < P2; ++q) {
                const int n = 2 * ((t + P2 * bb) + P1 * q);
                const C va = st[n + (sw ? 1 : 0)], vb = st[n + (sw ? 0 : 1)];
                o0[bb][q].x = sw ? vb.x : va.x; o0[bb][q].y = sw ? vb.y : va.y;
                o1[bb][q].x = sw ? va.x : vb.x; o1[bb][q].y = sw ? va.y : vb.y;
            }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp(); // every lane has its values: the landing zone may be refilled
    };
    // V(r) of x task u (vloc)
    auto v_load = [&](const PlaneTask &tk, int u, T (&v0)[B2][P2], T (&v1)[B2][P2]) {
        const int yl = (warp + u * NW) * G + f;
        const T *vrow = vloc + ((long long)tk.z * N + (2 * yl + tk.r)) * N;
#pragma unroll
        for (int bb = 0; bb < B2; ++bb)
#pragma unroll
            for (int q = 0; q < P2; ++q) {
                const int n = 2 * ((t + P2 * bb) + P1 * q);
                v0[bb][q] = __ldg(vrow + n);
                v1[bb][q] = __ldg(vrow + n + 1);
            }
    };

    // ---- stage bodies ------------------------------------------------------------------------------
    // inverse y pass of one column group: stick values -> column of the plane buffer
    auto yinv_body = [&](C (&x)[P1], C bv, const YCol &c, int r, C *pbuf) {
        if (r == 0) {
            x[P1 / 2] = cadd(x[P1 / 2], bv);
        } else {
            x[P1 / 2] = csub(x[P1 / 2], bv);
            pre_inv<F, 0, T>(x, g);
        }
        C y[B2][P2];
        sub_inv<F, T>(x, y, tws, ex, t);
        if (c.act) {
            C *pc = pbuf + c.col * YP;
#pragma unroll
            for (int bb = 0; bb < B2; ++bb)
#pragma unroll
                for (int q = 0; q < P2; ++q) pc[(t + P2 * bb) + P1 * q] = y[bb][q];
        }
    };
    // forward y pass of one column group: column of the plane buffer -> partial A of residue r
    auto yfwd_body = [&](const YCol &c, int r, C *pbuf, C *dst) {
        C *pc = pbuf + c.col * YP;
        C y[B2][P2], x[P1];
#pragma unroll
        for (int bb = 0; bb < B2; ++bb)
#pragma unroll
            for (int q = 0; q < P2; ++q) y[bb][q] = pc[(t + P2 * bb) + P1 * q];
        if constexpr (MODE == MODE_FWD) sub_fwd<F, T>(y, x, tws, ExSkew<T, P2, 1>{pc, c.act}, t); // in place in the column
        else sub_fwd<F, T>(y, x, tws, ex, t);
        if (r != 0) post_fwd<F, 0, T>(x, g); // partial of residue 1: conj(W^{k_s}) G[k]
        if (c.act) {
            C *d = dst + c.co.x;
            const int idb = M / 2 - c.co.z;
            if (l0 && (unsigned)idb < (unsigned)c.co.y) d[idb] = r ? mk<T>(-x[P1 / 2].x, -x[P1 / 2].y) : x[P1 / 2];
#pragma unroll
            for (int j = 0; j < P1; ++j) {
                const int idx = ks_of<F>(t, j) - c.co.z;
                if ((unsigned)idx < (unsigned)c.co.y) d[idx] = x[j];
            }
        }
    };
    // inverse x pass of one line per group: plane buffer -> the line's values x = 2 n' + e in (o0, o1)
    auto xinv_body = [&](const C *pbuf, int yl, C (&o0)[B2][P2], C (&o1)[B2][P2]) {
        C x[P1], xs[P1];
#pragma unroll
        for (int j = 0; j < P1; ++j) {
            const int c = ks_of<F>(t, j) - k1lo;
            x[j] = (unsigned)c < (unsigned)nx ? pbuf[c * YP + yl] : czero<T>();
        }
        const int cb = M / 2 - k1lo;
        const C bv = (l0 && (unsigned)cb < (unsigned)nx) ? pbuf[cb * YP + yl] : czero<T>();
#pragma unroll
        for (int j = 0; j < P1; ++j) xs[j] = x[j];
        xs[P1 / 2] = cadd(xs[P1 / 2], bv);
        sub_inv<F, T>(xs, o0, tws, ex, t);
        x[P1 / 2] = csub(x[P1 / 2], bv);
        pre_inv<F, 0, T>(x, g);
        sub_inv<F, T>(x, o1, tws, ex, t);
    };
    // forward x pass of one line per group: (o0, o1) -> the occupied k1 columns of the plane buffer
    auto xfwd_body = [&](C (&o0)[B2][P2], C (&o1)[B2][P2], C *pbuf, int yl) {
        C g0[P1], g1[P1];
        if constexpr (MODE == MODE_FWD) {
            // exchanged in place in the line's own (still unused) slots of the plane buffer
            sub_fwd<F, T>(o0, g0, tws, ExSkew<T, P2, YP>{pbuf + yl, true}, t);
            sub_fwd<F, T>(o1, g1, tws, ExSkew<T, P2, YP>{pbuf + yl, true}, t);
            __syncwarp();
        } else {
            sub_fwd<F, T>(o0, g0, tws, ex, t);
            sub_fwd<F, T>(o1, g1, tws, ex, t);
        }
        post_fwd<F, 0, T>(g1, g);
        const int cb = M / 2 - k1lo;
        if (l0 && (unsigned)cb < (unsigned)nx) pbuf[cb * YP + yl] = csub(g0[P1 / 2], g1[P1 / 2]);
#pragma unroll
        for (int j = 0; j < P1; ++j) {
            const int c = ks_of<F>(t, j) - k1lo;
            if ((unsigned)c < (unsigned)nx) pbuf[c * YP + yl] = cadd(g0[j], g1[j]);
        }
    };

    // ---- prefetch registers and the task records of iterations it-2 .. it+1 --------------------------
    T vq0[B2][P2], vq1[B2][P2];            // V(r) of the next x task (VLOC)
    PlaneTask tkPP = {0, 0, 0}, tkP = {0, 0, 0}, tkC = decode(0), tkN = decode(1);
    if (tid == 0) {
        mbar_init(&bar_full, 1);
        mbar_init(&bar_empty, NW);
        for (int w = 0; w < NW; ++w) mbar_init(&bar_line[w], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (ktasks > 0) {
        if constexpr (MODE != MODE_FWD) {
            if (tid == 0) stage_issue(tkC);
        } else {
            line_issue(tkC, 0);
        }
        if constexpr (MODE == MODE_VLOC) v_load(tkC, 0, vq0, vq1);
    }

#pragma unroll 1
    for (int it = 0; it < ktasks + LAG; tkPP = tkP, tkP = tkC, tkC = tkN, tkN = decode(it + 2), ++it) {
        // ============================================================ forward x pass of task it -> buf[it&1]
        if constexpr (MODE == MODE_FWD) {
            if (it < ktasks) {
                C *pbuf = pbuf0 + (it & 1) * PB;
#pragma unroll
                for (int u = 0; u < XT; ++u) {
                    C o0[B2][P2], o1[B2][P2];
                    line_read(o0, o1);
                    // the next x task's lines land while this one is transformed
                    if (u + 1 < XT) line_issue(tkC, u + 1);
                    else if (it + 1 < ktasks) line_issue(tkN, 0);
                    xfwd_body(o0, o1, pbuf, (warp + u * NW) * G + f);
                }
            }
        }
        // ============================================================ forward y pass: buf -> partial A
        if constexpr (MODE != MODE_INV) {
            const int k = it - LAG;
            if (k >= 0) {
                const PlaneTask tk = (LAG == 1) ? tkP : tkPP;
                C *pbuf = pbuf0 + (k & 1) * PB;
                C *dst = Aout + (long long)tk.b * a_out_stride + ((long long)tk.r * pl.n3 + tk.z) * pl.pitch;
#pragma unroll
                for (int u = 0; u < YT; ++u)
                    if (warp + u * NW < ntask_y) yfwd_body(yc[u], tk.r, pbuf, dst);
                for (int task = warp + YT * NW; task < ntask_y; task += NW) yfwd_body(ycol(task), tk.r, pbuf, dst);
                // single-stick columns: one warp per column, dot product with conj(W^{k2 y})
                for (int i = warp; i < n_one; i += NW) {
                    const int col = ct.perm[pl.n_multi + i];
                    const int4 co = ct.col[col];
                    C acc = czero<T>();
                    for (int yl = lane; yl < M; yl += 32)
                        acc = cadd(acc, cmulc(pbuf[col * YP + yl], tw[modn<N>(co.z * (2 * yl + tk.r))]));
#pragma unroll
                    for (int sft = 16; sft > 0; sft >>= 1) {
                        acc.x += __shfl_xor_sync(0xffffffffu, acc.x, sft);
                        acc.y += __shfl_xor_sync(0xffffffffu, acc.y, sft);
                    }
                    if (lane == 0) dst[co.x] = acc;
                }
            }
        }
        if constexpr (MODE != MODE_FWD) {
            // ======================================================== inverse y pass of task it -> buf[it&1]
            if (it < ktasks) {
                C *pbuf = pbuf0 + (it & 1) * PB;
                mbar_wait(&bar_full, it & 1); // the row of task it has landed
                for (int task = warp; task < ntask_y; task += NW) {
                    const YCol c = (task == warp) ? yc[0] : (task == warp + NW) ? yc[1] : ycol(task);
                    C x[P1], bv;
                    yinv_load(c, x, bv);
                    yinv_body(x, bv, c, tkC.r, pbuf);
                }
                // single-stick columns (same warp as in the forward pass): closed form x W^{k2 y}
                for (int i = warp; i < n_one; i += NW) {
                    const int col = ct.perm[pl.n_multi + i];
                    const int4 co = ct.col[col];
                    const C v = stage[co.x];
                    __syncwarp();
                    for (int yl = lane; yl < M; yl += 32) pbuf[col * YP + yl] = cmul(v, tw[modn<N>(co.z * (2 * yl + tkC.r))]);
                }
                // this warp no longer reads the staged row; when all have said so, the next row may land:
                // it is in flight during the whole x pass below
                __syncwarp();
                if (lane == 0) mbar_arrive(&bar_empty);
                if (tid == 0 && it + 1 < ktasks) {
                    mbar_wait(&bar_empty, it & 1);
                    stage_issue(tkN);
                }
            }
            // ======================================================== x pass of task it-1 in buf[(it-1)&1]
            if (it >= 1 && it - 1 < ktasks) {
                C *pbuf = pbuf0 + ((it - 1) & 1) * PB;
#pragma unroll
                for (int u = 0; u < XT; ++u) {
                    const int yl = (warp + u * NW) * G + f;
                    C o0[B2][P2], o1[B2][P2];
                    xinv_body(pbuf, yl, o0, o1);
                    if constexpr (MODE == MODE_INV) {
                        C *row = cub_out + (((long long)tkP.b * pl.n3 + tkP.z) * N + (2 * yl + tkP.r)) * N;
#pragma unroll
                        for (int bb = 0; bb < B2; ++bb)
#pragma unroll
                            for (int q = 0; q < P2; ++q) st_pair(row + 2 * ((t + P2 * bb) + P1 * q), o0[bb][q], o1[bb][q]);
                    } else {
#pragma unroll
                        for (int bb = 0; bb < B2; ++bb)
#pragma unroll
                            for (int q = 0; q < P2; ++q) {
                                o0[bb][q].x *= vq0[bb][q]; o0[bb][q].y *= vq0[bb][q];
                                o1[bb][q].x *= vq1[bb][q]; o1[bb][q].y *= vq1[bb][q];
                            }
                        // V(r) of the next x task is in flight during the forward half
                        if (u + 1 < XT) v_load(tkP, u + 1, vq0, vq1);
                        else if (it < ktasks) v_load(tkC, 0, vq0, vq1);
                        xfwd_body(o0, o1, pbuf, yl);
                    }
                }
            }
        }
        __syncthreads();
    }
}

} // namespace fftb
