// fftb_plane_pf.cuh -- persistent plane kernel of the fast path (sm_100a).
//
// Same mathematics and the same building blocks as fftb_plane_fast.cuh (half-band line = two length-M
// transforms, each done by a group of P2 lanes around one exchange; PAPER.md:96 Fig. 3, :112 staged
// padding).  This file is the schedule:
//   * persistent grid, CTA c owns the z-planes c, c + G, ... of the batch; a plane is processed whole:
//     its two y residues r = 0, 1 live in the two plane buffers pbuf[r][column][y'] in shared memory.
//       INV   Y: row A[b][z][.] -> both residues of every occupied k1 column      | barrier
//             X: 128 lines (buffer y&1, row y>>1) -> cuboid                        | barrier
//       FWD   X: cuboid lines -> occupied k1 columns of pbuf[y&1]                  | barrier
//             Y: columns of both buffers -> G_0 + conj(W^k) G_1 -> A[b][z][.]      | barrier
//       VLOC  Y_inv | barrier | X: inverse, V(r), forward in place | barrier | Y_fwd (then the Y_inv of the
//             next plane on the same columns by the same warp, no barrier in between)
//     The barrier in front of a plane's FIRST phase (INV: after the x pass, FWD: after the y pass) is SPLIT: a warp arrives on an
//     mbarrier when it is done and waits only where its next task first touches the plane buffers -- after the task's inputs
//     have been read and the register-only front of its transforms is done (ncu: a quarter of the inverse kernel's stall
//     samples sat behind the two CTA barriers; 0.966 -> 0.94 ms inverse, 1.025 -> 1.015 ms forward on config 3).
//   * every exchange of a transform is done IN PLACE in the line or column of the plane buffer it
//     works on (ExSkew), so the only other shared memory is the TMA landing zone.
//   * global memory is read by the TMA engine only (cp.async.bulk + mbarrier), one plane / one x task
//     ahead of its use: the row of A as one bulk copy per plane, the G consecutive cuboid lines of an x
//     task as one bulk copy per warp.  Measured on B200: register prefetch over the same distance keeps a
//     scoreboard slot busy, and every later wait on that slot waits for the prefetch too; occupancy
//     cannot hide the latency either, because complex128 butterflies need far more than 64 registers.
//   * 8 warps x up to 255 registers per CTA: the transform core alone already reaches the FP64 pipe's
//     rate with 8 warps per SM (79 clk per four 64-point transforms against a floor of 75).
#pragma once
#include "fftb_plane_fast.cuh"

namespace fftb {

template <typename T, class F, int NW> struct PlanePF {
    // elements of one plane buffer (one y residue).  The two buffers hold the even and the odd lines, and a
    // shared-memory wavefront covers GW = LW / P2 lane groups = lines y, y+1 (one row of BOTH buffers), y+2, ...:
    // with YP congruent to GW (FastCfg) the buffers must be GW/2 apart modulo LW for those accesses to
    // fall into different banks (complex64, and complex128 with 4 lanes per transform)
    static constexpr int GW = F::LW / F::P2;
    static constexpr int PB0 = F::NCOL * F::YP;
    static constexpr int PB = GW < 2 ? PB0 : PB0 + ((GW / 2 - PB0 % F::LW) + F::LW) % F::LW;
    static constexpr int NXT = F::N / F::G;    // x tasks per plane (G consecutive lines each)
    static constexpr int XT = NXT / NW;        // x tasks per warp and plane
    static_assert(NXT % NW == 0 && XT >= 1, "x tasks must divide evenly over the warps");
    // two plane buffers + the TMA landing zone: one row of A (pitch elements) for INV and VLOC, G cuboid
    // lines per warp for FWD
    static size_t smem_bytes_mode(int mode, int pitch)
    {
        return sizeof(cx<T>) * (2 * (size_t)PB + (mode == MODE_FWD ? (size_t)NW * F::G * F::N : (size_t)pitch));
    }
};


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
// ask for `bytes` (a multiple of 16) at gsrc to be brought into L2; no completion is signalled
__device__ __forceinline__ void bulk_prefetch_l2(const void *gsrc, unsigned bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(gsrc), "r"(bytes) : "memory");
}

template <typename T, class F, int NW, int MODE>
__global__ void __launch_bounds__(NW * 32, 1)
plane_pf_k(const __grid_constant__ DevPlan pl, const __grid_constant__ ColTab ct, const cx<T> *__restrict__ Ain,
           cx<T> *__restrict__ Aout, const cx<T> *__restrict__ cub_in, cx<T> *__restrict__ cub_out,
           const T *__restrict__ vloc, long long a_in_stride, long long a_out_stride, int nplanes)
{
    using C = cx<T>;
    using PF = PlanePF<T, F, NW>;
    constexpr int N = F::N, M = F::M, P1 = F::P1, P2 = F::P2, B2 = F::B2, G = F::G, YP = F::YP;
    constexpr int PB = PF::PB, XT = PF::XT;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C *pbuf0 = reinterpret_cast<C *>(smem_raw); // [2 residues][NCOL][YP]: column c = k1 - k1lo, local line y'
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int f = lane / P2, t = lane % P2;
    C *stage = pbuf0 + 2 * PB;                      // INV, VLOC: landing zone of the row A[b][z][0..pitch)
    C *lstage = pbuf0 + 2 * PB + warp * (G * N);    // FWD: landing zone of this warp's next x task (G lines)
    __shared__ __align__(8) unsigned long long bar_full, bar_line[NW], bar_pb;
    unsigned pb_par = 0;
    bool pb_pending = false; // this warp has arrived on bar_pb and not waited yet
    const unsigned stage_bytes = (unsigned)pl.pitch * (unsigned)sizeof(C);
    unsigned line_par = 0;
    const C *tw = reinterpret_cast<const C *>(pl.tw1); // N1 == N2: one table
    C tws[P1];
#pragma unroll
    for (int m = 1; m < P1; ++m) tws[m] = tw[modn<N>(2 * t * m)];
    tws[0] = mk<T>((T)1, (T)0);
    const C g = tw[t];
    const int nx = pl.nxocc, k1lo = pl.k1lo;
    const bool l0 = (t == 0);
    const int n_one = nx - pl.n_multi;
    const int ntask_y = ycol_tasks<F>(pl.n_multi);
    const int kplanes = nplanes > (int)blockIdx.x ? (nplanes - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;

    // column group of this lane in y task `task`
    struct YCol { bool act; int col; int4 co; };
    auto ycol = [&](int task) -> YCol {
        YCol c;
        const int ci = ycol_index<F>(task, f);
        c.act = task < ntask_y && ci < pl.n_multi;
        c.col = ct.perm[c.act ? ci : 0];
        c.co = ct.col[c.col];
        return c;
    };
    const YCol yc0 = ycol(warp), yc1 = ycol(warp + NW); // the warp's usual two tasks, looked up once
    auto ycol_of = [&](int task) -> YCol { return task == warp ? yc0 : task == warp + NW ? yc1 : ycol(task); };

    // ---- asynchronous loads ------------------------------------------------------------------------
    // one thread asks the TMA engine for the row of plane (b, z); completion is signalled on bar_full
    auto stage_issue = [&](int b, int z) {
        mbar_expect_tx(&bar_full, stage_bytes);
        bulk_load(stage, Ain + (long long)b * a_in_stride + (long long)z * pl.pitch, stage_bytes, &bar_full);
    };
    // the G consecutive cuboid lines y = v G .. v G + G - 1 of x task v are one contiguous block
    auto line_issue = [&](int b, int z, int v) {
        if (lane == 0) {
            mbar_expect_tx(&bar_line[warp], (unsigned)(G * N * sizeof(C)));
            bulk_load(lstage, cub_in + (((long long)b * pl.n3 + z) * N + (long long)v * G) * N, (unsigned)(G * N * sizeof(C)),
                      &bar_line[warp]);
        }
    };
    // ... read from there as (x, x+1) pairs; half of the lanes take the odd element first so that the
    // 32-byte-strided 16-byte reads of a quarter warp fall into different bank groups
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
    // V(r) of x task v (vloc), one task ahead in registers (L2 resident, 16 values per lane)
    auto v_load = [&](int z, int v, T (&v0)[B2][P2], T (&v1)[B2][P2]) {
        const T *vrow = vloc + ((long long)z * N + (v * G + f)) * N;
#pragma unroll
        for (int bb = 0; bb < B2; ++bb)
#pragma unroll
            for (int q = 0; q < P2; ++q) {
                const int n = 2 * ((t + P2 * bb) + P1 * q);
                v0[bb][q] = __ldg(vrow + n);
                v1[bb][q] = __ldg(vrow + n + 1);
            }
    };

    // split barrier in front of a plane's first phase: the other warps are done with the plane buffers
    auto pb_wait = [&]() {
        if (pb_pending) {
            mbar_wait(&bar_pb, pb_par);
            pb_par ^= 1u;
            pb_pending = false;
        }
    };
    auto pb_arrive = [&]() {
        asm volatile("mbarrier.arrive.release.cta.shared::cta.b64 _, [%0];" ::"r"(smem_u32(&bar_pb)) : "memory");
        pb_pending = true;
    };
    // ---- stage bodies ------------------------------------------------------------------------------
    C *const pb0 = pbuf0, *const pb1 = pbuf0 + PB;
    // inverse y pass of one column group: stick values (staged row) -> the column in both residue buffers
    auto yinv_body = [&](const YCol &c) {
        const C *src = stage + c.co.x;
        C x[P1], xs[P1], y[B2][P2];
#pragma unroll
        for (int j = 0; j < P1; ++j) {
            const int idx = ks_of<F>(t, j) - c.co.z;
            x[j] = (c.act && (unsigned)idx < (unsigned)c.co.y) ? src[idx] : czero<T>();
        }
        const int idb = M / 2 - c.co.z;
        const C bv = (c.act && l0 && (unsigned)idb < (unsigned)c.co.y) ? src[idb] : czero<T>();
#pragma unroll
        for (int j = 0; j < P1; ++j) xs[j] = x[j];
        xs[P1 / 2] = cadd(xs[P1 / 2], bv);
        C *pc = pb0 + c.col * YP;
        sub_inv_front<F, T>(xs, tws);
        x[P1 / 2] = csub(x[P1 / 2], bv);
        pre_inv<F, 0, T>(x, g);
        sub_inv_front<F, T>(x, tws);
        pb_wait(); // INV: the previous plane's x pass is over in every warp
        sub_inv_back<F, T>(xs, y, ExSkew<T, P2, 1>{pc, c.act}, t); // exchanged in place in the destination column
        __syncwarp();
        if (c.act) {
#pragma unroll
            for (int bb = 0; bb < B2; ++bb)
#pragma unroll
                for (int q = 0; q < P2; ++q) pc[(t + P2 * bb) + P1 * q] = y[bb][q];
        }
        pc = pb1 + c.col * YP;
        sub_inv_back<F, T>(x, y, ExSkew<T, P2, 1>{pc, c.act}, t);
        __syncwarp();
        if (c.act) {
#pragma unroll
            for (int bb = 0; bb < B2; ++bb)
#pragma unroll
                for (int q = 0; q < P2; ++q) pc[(t + P2 * bb) + P1 * q] = y[bb][q];
        }
    };
    // forward y pass of one column group: the column of both residue buffers -> A
    auto yfwd_body = [&](const YCol &c, C *dst) {
        C *pc0 = pb0 + c.col * YP, *pc1 = pb1 + c.col * YP;
        C y[B2][P2], x0[P1], x1[P1];
#pragma unroll
        for (int bb = 0; bb < B2; ++bb)
#pragma unroll
            for (int q = 0; q < P2; ++q) y[bb][q] = pc0[(t + P2 * bb) + P1 * q];
        sub_fwd<F, T>(y, x0, tws, ExSkew<T, P2, 1>{pc0, c.act}, t); // exchanged in place in the column
#pragma unroll
        for (int bb = 0; bb < B2; ++bb)
#pragma unroll
            for (int q = 0; q < P2; ++q) y[bb][q] = pc1[(t + P2 * bb) + P1 * q];
        sub_fwd<F, T>(y, x1, tws, ExSkew<T, P2, 1>{pc1, c.act}, t);
        post_fwd<F, 0, T>(x1, g); // the part of residue 1: conj(W^{k_s}) G_1[k]
        if (c.act) {
            C *d = dst + c.co.x;
            const int idb = M / 2 - c.co.z;
            if (l0 && (unsigned)idb < (unsigned)c.co.y) d[idb] = csub(x0[P1 / 2], x1[P1 / 2]);
#pragma unroll
            for (int j = 0; j < P1; ++j) {
                const int idx = ks_of<F>(t, j) - c.co.z;
                if ((unsigned)idx < (unsigned)c.co.y) d[idx] = cadd(x0[j], x1[j]);
            }
        }
    };
    // inverse x pass of one line per group: plane buffer -> the line's values x = 2 n' + e in (o0, o1)
    auto xinv_body = [&](C *pbuf, int yl, C (&o0)[B2][P2], C (&o1)[B2][P2]) {
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
        // the line's slots are dead once every lane holds its inputs: both exchanges happen in them
        sub_inv<F, T>(xs, o0, tws, ExSkew<T, P2, YP>{pbuf + yl, true}, t);
        x[P1 / 2] = csub(x[P1 / 2], bv);
        pre_inv<F, 0, T>(x, g);
        sub_inv<F, T>(x, o1, tws, ExSkew<T, P2, YP>{pbuf + yl, true}, t);
    };
    // forward x pass of one line per group: (o0, o1) -> the occupied k1 columns of the plane buffer
    auto xfwd_body = [&](C (&o0)[B2][P2], C (&o1)[B2][P2], C *pbuf, int yl) {
        C g0[P1], g1[P1];
        sub_fwd_front<F, T>(o0, tws);
        sub_fwd_front<F, T>(o1, tws);
        pb_wait(); // FWD: the previous plane's y pass is over in every warp
        // exchanged in place in the line's own slots (unused so far in FWD, dead after the inverse half in VLOC)
        sub_fwd_back<F, T>(o0, g0, ExSkew<T, P2, YP>{pbuf + yl, true}, t);
        sub_fwd_back<F, T>(o1, g1, ExSkew<T, P2, YP>{pbuf + yl, true}, t);
        __syncwarp();
        post_fwd<F, 0, T>(g1, g);
        const int cb = M / 2 - k1lo;
        if (l0 && (unsigned)cb < (unsigned)nx) pbuf[cb * YP + yl] = csub(g0[P1 / 2], g1[P1 / 2]);
#pragma unroll
        for (int j = 0; j < P1; ++j) {
            const int c = ks_of<F>(t, j) - k1lo;
            if ((unsigned)c < (unsigned)nx) pbuf[c * YP + yl] = cadd(g0[j], g1[j]);
        }
    };
    // single-stick columns, one warp per column.  Inverse: closed form x W^{k2 y}; forward: dot product.
    auto yinv_single = [&]() {
        if constexpr (MODE == MODE_INV) {
            // the (column, y) pairs are dealt over ALL threads of the CTA: a warp per column would leave the other warps waiting
            // at the barrier behind this phase (two such columns for a sphere: about 350 cycles per plane on two of eight warps)
            for (int it = tid; it < n_one * N; it += NW * 32) {
                const int i = it / N, y = it % N;
                const int col = ct.perm[pl.n_multi + i];
                const int4 co = ct.col[col];
                (y & 1 ? pb1 : pb0)[col * YP + (y >> 1)] = cmul(stage[co.x], tw[modn<N>(co.z * y)]);
            }
        } else {
            // VLOC: a column belongs to ONE warp from the forward y pass of a plane through the inverse y pass of the next
            // (there is no barrier in between)
            for (int i = warp; i < n_one; i += NW) {
                const int col = ct.perm[pl.n_multi + i];
                const int4 co = ct.col[col];
                const C v = stage[co.x];
                for (int y = lane; y < N; y += 32) (y & 1 ? pb1 : pb0)[col * YP + (y >> 1)] = cmul(v, tw[modn<N>(co.z * y)]);
            }
        }
    };
    auto yfwd_single = [&](C *dst) {
        for (int i = warp; i < n_one; i += NW) {
            const int col = ct.perm[pl.n_multi + i];
            const int4 co = ct.col[col];
            C acc = czero<T>();
            for (int y = lane; y < N; y += 32) acc = cadd(acc, cmulc((y & 1 ? pb1 : pb0)[col * YP + (y >> 1)], tw[modn<N>(co.z * y)]));
#pragma unroll
            for (int sft = 16; sft > 0; sft >>= 1) {
                acc.x += __shfl_xor_sync(0xffffffffu, acc.x, sft);
                acc.y += __shfl_xor_sync(0xffffffffu, acc.y, sft);
            }
            if (lane == 0) dst[co.x] = acc;
        }
    };

    // ---- the persistent loop over this CTA's planes --------------------------------------------------
    if (tid == 0) {
        mbar_init(&bar_full, 1);
        mbar_init(&bar_pb, NW * 32);
        for (int w = 0; w < NW; ++w) mbar_init(&bar_line[w], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    T vq0[B2][P2], vq1[B2][P2]; // V(r) of the next x task (VLOC)
    int z = blockIdx.x % pl.n3, b = blockIdx.x / pl.n3;          // current plane
    const int dz = gridDim.x % pl.n3, db = gridDim.x / pl.n3;      // step to this CTA's next plane
    if (kplanes > 0) {
        if constexpr (MODE == MODE_FWD) line_issue(b, z, warp);
        else if (tid == 0) stage_issue(b, z);
        if constexpr (MODE == MODE_VLOC) v_load(z, warp, vq0, vq1);
    }
#pragma unroll 1
    for (int i = 0; i < kplanes; ++i) {
        const int zc = z + dz, zn = zc >= pl.n3 ? zc - pl.n3 : zc, bn = b + db + (zc >= pl.n3 ? 1 : 0); // next plane
        const bool more = i + 1 < kplanes;
        if constexpr (MODE != MODE_FWD) {
            // ======================================================== inverse y pass: staged row -> both buffers
            mbar_wait(&bar_full, i & 1);
            for (int task = warp; task < ntask_y; task += NW) yinv_body(ycol_of(task));
            pb_wait(); // a warp without a y task
            yinv_single();
            __syncthreads();
            // nobody reads the staged row any more: the next plane's row lands during the x pass
            if (tid == 0 && more) stage_issue(bn, zn);
            // ======================================================== x pass: line y of buffer y&1, row y>>1
#pragma unroll
            for (int u = 0; u < XT; ++u) {
                const int v = warp + u * NW, y = v * G + f;
                C *pbuf = (y & 1) ? pb1 : pb0;
                C o0[B2][P2], o1[B2][P2];
                xinv_body(pbuf, y >> 1, o0, o1);
                if constexpr (MODE == MODE_INV) {
                    C *row = cub_out + (((long long)b * pl.n3 + z) * N + y) * N;
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
                    if (u + 1 < XT) v_load(z, v + NW, vq0, vq1);
                    else if (more) v_load(zn, warp, vq0, vq1);
                    xfwd_body(o0, o1, pbuf, y >> 1);
                }
            }
            if constexpr (MODE == MODE_INV) pb_arrive(); // split: waited for inside the next plane's first y task
            else __syncthreads();
        } else {
            // ======================================================== forward x pass: cuboid lines -> buffers
#pragma unroll
            for (int u = 0; u < XT; ++u) {
                const int v = warp + u * NW, y = v * G + f;
                C o0[B2][P2], o1[B2][P2];
                line_read(o0, o1);
                // the next x task's lines land while this one is transformed
                if (u + 1 < XT) line_issue(b, z, v + NW);
                else if (more) line_issue(bn, zn, warp);
                xfwd_body(o0, o1, (y & 1) ? pb1 : pb0, y >> 1);
            }
            __syncthreads();
        }
        if constexpr (MODE != MODE_INV) {
            // ======================================================== forward y pass: both buffers -> A
            C *dst = Aout + (long long)b * a_out_stride + (long long)z * pl.pitch;
            for (int task = warp; task < ntask_y; task += NW) yfwd_body(ycol_of(task), dst);
            yfwd_single(dst);
            // FWD: the next plane's x pass overwrites the buffers.  VLOC: the next plane's inverse y pass
            // touches the same columns from the same warp, no barrier needed.
            if constexpr (MODE == MODE_FWD) pb_arrive(); // split: waited for inside the next plane's first x task
        }
        z = zn; b = bn;
    }
}

} // namespace fftb
