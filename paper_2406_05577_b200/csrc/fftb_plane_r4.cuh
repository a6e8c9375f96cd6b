// fftb_plane_r4.cuh -- persistent inverse plane kernel for grids of 4 x 64 = 256 points per axis (sm_100a).
//
// The 256^3 / radius-64 problem is the paper's own workload shape ("256^3 grid ... sphere
// diameter 128").  A z-plane of both y residues (532 KB in complex128) does not fit the schedule of
// fftb_plane_pf.cuh, so the half-band axis is split FOUR ways instead of two: with n = 4 n' + e,
//     out[4 n' + e] = sum_k (x[k] W^{e k}) w_64^{k n'},   W = exp(2 pi j / 256),  k in [-64, 64],
// i.e. four length-64 transforms u_e of the input folded onto 64 slots: slot s = k mod 64 receives
// b = x[s] and a = x[s - 64] (and slot 0 the alias c = x[+64]):
//     u_e[s] = W^{e s} (b + (-j)^e a)  [+ (+j)^e c for s = 0].
// e = 0 costs one addition per slot, the others one complex multiplication more: 15% more FP64 work
// than a two-level split, but every transform is the 8 x 8 length-64 core of fftb_plane_fast.cuh and a
// QUARTER plane (129 columns x 64 lines, 134 KB) fits in shared memory next to the TMA landing zones.
//
// Schedule: persistent grid, CTA c owns the planes c, c + G, ...; per plane four quarters r = 0..3:
//     Y_r: every occupied k1 column -> u_r -> length-64 transform -> pbuf[column][y'] (y = 4 y' + r) | barrier
//     X_r: each of the 64 lines y = 4 y' + r: 129 inputs read once, four folded transforms, 64-byte
//          runs (x = 4 n' .. 4 n' + 3) stored as two 32-byte stores                                  | barrier
// The stick values of a column group arrive by TMA bulk copies in a per-warp landing zone, one y task
// ahead (cp.async.bulk + mbarrier); the row of A is read four times per plane, from L2.
// plane_r4_fwd_k below is the adjoint chain, plane_r4_vloc_k the fused local-potential apply.
#pragma once
#include "fftb_plane_pf.cuh"
#include "fftb_tmem.cuh"
#include <cuda.h>

namespace fftb {

constexpr int R4_MAXCOL = 129;
struct ColTab4 {
    int4 col[R4_MAXCOL]; // {first stick, stick count, k2lo, 0} per occupied k1 column
    int perm[R4_MAXCOL]; // multi-stick columns first, then the single-stick ones
};

template <typename T, int NW> struct PlaneR4 {
    using F = FastCfg<T, 128, 8, 8>;              // the length-64 core: 8 lanes x 8 values
    static constexpr int N = 256, M = 64;
    static constexpr int NCOL = 2 * M + 1, YP = F::YP;
    static constexpr int PB = NCOL * YP;          // one quarter plane
    static constexpr int ZCOL = 2 * M + 4;        // landing zone pitch per column (129 values + alignment slack, 16-byte multiple)
    static constexpr int ZONE = F::G * ZCOL;      // per warp: the G columns of its next y task (>= LZE: also a staging area, plane_r4_inv_k)
    static constexpr int NXT = M / F::G;          // x tasks per quarter (G lines each)
    static_assert(NXT % NW == 0, "x tasks must divide evenly over the warps");
    static constexpr size_t smem_bytes = sizeof(cx<T>) * ((size_t)PB + (size_t)NW * ZONE) + 128; // + alignment slack of the zones
    // y tasks (G columns each) per quarter: at most ycol_tasks(NCOL), dealt round-robin over the warps
    static constexpr int MAXT = (((NCOL + 7) / 8 * 8 + F::G - 1) / F::G + NW - 1) / NW;
    // y tasks per warp whose partial sums fit the warp's share of tensor memory (two warps per lane quarter: 256 columns)
    static constexpr int TMT = 256 / tmem_cols16<T>();
    // forward kernel: elements of a warp's landing zone (G lines x 64 (x, x+1) pairs) and its dynamic shared memory
    static constexpr int LZE = F::G * M * 2;
    static constexpr size_t smem_bytes_fwd = sizeof(cx<T>) * ((size_t)PB + (size_t)NW * LZE) + 128;
};

// The y tasks of a warp are the same for every plane and quarter: which column each lane group works on and, for the
// kernels that read the row of A, which bulk copies bring the task's stick runs into the warp's landing zone.  Looked up
// ONCE per kernel and kept in shared memory -- inside the plane loop a task then costs one shared-memory load instead
// of two dependent look-ups in the column tables, a warp reduction and up to G copy instructions (measured on config 5:
// 740 of the 2 400 cycles of an inverse y task).
template <typename T, int NW> struct R4Tasks {
    using R4 = PlaneR4<T, NW>;
    static constexpr int G = R4::F::G;
    int4 desc[NW][R4::MAXT][G]; // {x, stick count (0: no column), k2lo, column}; x = first value of the column in the landing
                                // zone (r4_tasks_zone) or first stick of the column in the row of A (r4_tasks_rows)
    int4 copy[NW][R4::MAXT][G]; // bulk copies of the task: {row offset, bytes (0: none), zone offset, .}; .w = first stick of this lane group's column in the row of A
    int total[NW][R4::MAXT];    // bytes of all copies of the task
};
template <typename T, int NW>
__device__ __forceinline__ void r4_tasks_rows(R4Tasks<T, NW> &ts, const DevPlan &pl, const ColTab4 &ct, int warp, int lane, int ytasks_w)
{
    using F = typename PlaneR4<T, NW>::F;
    for (int k = 0; k < ytasks_w; ++k) {
        if (lane < F::G) {
            const int ci = ycol_index<F>(warp + k * NW, lane);
            int4 d = make_int4(0, 0, 0, 0);
            if (ci < pl.n_multi) {
                const int col = ct.perm[ci];
                const int4 co = ct.col[col];
                d = make_int4(co.x, co.y, co.z, col);
            }
            ts.desc[warp][k][lane] = d;
        }
    }
    __syncwarp();
}
// If the G columns of a task are neighbours in k1 (complex128: ycol_index is the identity) their stick runs are ONE
// contiguous range of the row -- the sticks are ordered by (k1, k2) -- and arrive as one copy, unless single-stick
// columns of an explicit map lie in between and make the range longer than the zone; otherwise one copy per column
// (complex64: 16-byte units, so a run is widened to even element indices; the row's pitch is even).
template <typename T, int NW>
__device__ __forceinline__ void r4_tasks_zone(R4Tasks<T, NW> &ts, const DevPlan &pl, const ColTab4 &ct, int warp, int lane, int ytasks_w)
{
    using R4 = PlaneR4<T, NW>;
    using F = typename R4::F;
    constexpr int G = F::G, EA = 16 / (int)sizeof(cx<T>);
    constexpr int GWy = F::LW / F::P2 < 1 ? 1 : F::LW / F::P2, Dy = F::P2 / GWy;
    constexpr bool NEIGHBOURS = (GWy <= 1 || Dy <= 1);
    for (int k = 0; k < ytasks_w; ++k) {
        int4 d = make_int4(0, 0, 0, 0), cp = make_int4(0, 0, 0, 0);
        int x1 = 0, col_first = 0;
        if (lane < G) {
            const int ci = ycol_index<F>(warp + k * NW, lane);
            if (ci < pl.n_multi) {
                const int col = ct.perm[ci];
                const int4 co = ct.col[col];
                d = make_int4(co.x, co.y, co.z, col);
                x1 = co.x + co.y;
                col_first = co.x;
            }
        }
        // lane 0's column is the first of the task (it always exists); the largest end closes the range
        const int first = __shfl_sync(0xffffffffu, d.x, 0);
        int last = x1;
#pragma unroll
        for (int sft = 1; sft < G; sft <<= 1) last = max(last, __shfl_xor_sync(0xffffffffu, last, sft));
        const int a0 = first & ~(EA - 1), a1 = (last + EA - 1) & ~(EA - 1);
        if (NEIGHBOURS && a1 - a0 <= R4::ZONE) {
            if (lane == 0) cp = make_int4(a0, (a1 - a0) * (int)sizeof(cx<T>), 0, 0);
            d.x = d.y > 0 ? d.x - a0 : 0;
        } else if (lane < G && d.y > 0) {
            const int sh = d.x & (EA - 1);
            cp = make_int4(d.x - sh, ((d.y + sh + EA - 1) & ~(EA - 1)) * (int)sizeof(cx<T>), lane * R4::ZCOL, 0);
            d.x = lane * R4::ZCOL + sh;
        }
        int total = cp.y;
#pragma unroll
        for (int sft = 1; sft < G; sft <<= 1) total += __shfl_xor_sync(0xffffffffu, total, sft);
        if (lane < G) { cp.w = col_first; ts.desc[warp][k][lane] = d; ts.copy[warp][k][lane] = cp; }
        if (lane == 0) ts.total[warp][k] = total;
    }
    __syncwarp();
}
// TMA: the stick runs of this warp's y task k of the plane whose row of A is `row` -> the warp's landing zone
template <typename T, int NW>
__device__ __forceinline__ void r4_zone_issue(const R4Tasks<T, NW> &ts, const cx<T> *row, cx<T> *zone, unsigned long long *bar, int warp, int lane, int k)
{
    if (lane == 0) mbar_expect_tx(bar, (unsigned)ts.total[warp][k]);
    __syncwarp();
    if (lane < R4Tasks<T, NW>::G) {
        const int4 cp = ts.copy[warp][k][lane];
        if (cp.y > 0) bulk_load(zone + cp.z, row + cp.x, (unsigned)cp.y, bar);
    }
}

// u_e of one lane: slots s = t + 8 j; a = x[s - 64], b = x[s], c = x[+64] (lane 0, slot 0 only, else 0)
template <int E, int J, typename T>
__device__ __forceinline__ void r4_fold_inv(const cx<T> (&a)[8], const cx<T> (&b)[8], cx<T> c, cx<T> (&u)[8], cx<T> wte)
{
    if constexpr (J < 8) {
        cx<T> v = cadd(b[J], mul_root<(32 - 8 * E) % 32, 32, +1, T>(a[J])); // (-j)^E a
        if constexpr (J == 0) v = cadd(v, mul_root<(8 * E) % 32, 32, +1, T>(c)); // (+j)^E c
        if constexpr (E > 0) v = mul_root<(E * J) % 32, 32, +1, T>(cmul(v, wte)); // W^{E (t + 8 J)}
        u[J] = v;
        r4_fold_inv<E, J + 1, T>(a, b, c, u, wte);
    }
}

// one half (h = 0: e = 0, 1; h = 1: e = 2, 3) of the (x, x+1) pairs of the G lines y = 4 (ylg mod 64 ..+G) + r of a plane:
// coordinates of the cuboid tensor of plane_r4_fwd_k (built by the launcher): {0, h, 0, r, ylg}, ylg = (band n3 + z) 64 + y / 4
__device__ __forceinline__ void r4_lines_box_load(void *sdst, const void *tmap, int half, int r, int ylg, unsigned long long *bar)
{
    asm volatile("cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5, %6}], [%7];" ::"r"(smem_u32(sdst)),
                 "l"(tmap), "r"(0), "r"(half), "r"(0), "r"(r), "r"(ylg), "r"(smem_u32(bar))
                 : "memory");
}

// the same box the other way: shared memory -> cuboid (plane_r4_inv_k; completion by bulk async-group)
__device__ __forceinline__ void r4_lines_box_store(const void *tmap, int half, int r, int ylg, const void *ssrc)
{
    asm volatile("cp.async.bulk.tensor.5d.global.shared::cta.tile.bulk_group [%0, {%1, %2, %3, %4, %5}], [%6];" ::"l"(tmap), "r"(0), "r"(half), "r"(0),
                 "r"(r), "r"(ylg), "r"(smem_u32(ssrc))
                 : "memory");
}

template <typename T, int NW, bool TM>
__global__ void __launch_bounds__(NW * 32, 1)
plane_r4_inv_k(const __grid_constant__ DevPlan pl, const __grid_constant__ ColTab4 ct, const cx<T> *__restrict__ Ain,
               cx<T> *__restrict__ cub_out, const __grid_constant__ CUtensorMap cmap, long long a_in_stride, int nplanes)
{
    using C = cx<T>;
    using R4 = PlaneR4<T, NW>;
    using F = typename R4::F;
    constexpr int N = R4::N, M = R4::M, P2 = F::P2, G = F::G, YP = R4::YP, ZCOL = R4::ZCOL;
    constexpr int XT = R4::NXT / NW;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C *pbuf = reinterpret_cast<C *>(smem_raw); // [NCOL][YP]: column c = k1 - k1lo, line y' of the current quarter
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int f = lane / P2, t = lane % P2;
    // landing zone of this warp's next y task; TM: also the staging area of its x tasks (a tensor copy's shared-memory side
    // must be 128-byte aligned)
    unsigned char *z_raw = smem_raw + sizeof(C) * (size_t)R4::PB;
    z_raw += (128u - (smem_u32(z_raw) & 127u)) & 127u;
    C *zone = reinterpret_cast<C *>(z_raw) + warp * R4::ZONE;
    __shared__ __align__(8) unsigned long long bar_zone[NW];
    unsigned zone_par = 0;
    const C *tw = reinterpret_cast<const C *>(pl.tw1); // exp(+2 pi j i / 256)
    C tws[8];
#pragma unroll
    for (int m = 1; m < 8; ++m) tws[m] = tw[(4 * t * m) & (N - 1)]; // w_64^{t m}
    tws[0] = mk<T>((T)1, (T)0);
    C wt[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) wt[e] = tw[e * t]; // W^{e t}
    const int nx = pl.nxocc, k1lo = pl.k1lo;
    const int n_one = nx - pl.n_multi;
    const int ntask_y = ycol_tasks<F>(pl.n_multi);
    const int kplanes = nplanes > (int)blockIdx.x ? (nplanes - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;
    const int ytasks_w = ntask_y > warp ? (ntask_y - warp + NW - 1) / NW : 0; // y tasks of this warp per quarter

    __shared__ R4Tasks<T, NW> ts;
    r4_tasks_zone<T, NW>(ts, pl, ct, warp, lane, ytasks_w);
    auto zone_issue = [&](const C *row, int k) { r4_zone_issue<T, NW>(ts, row, zone, &bar_zone[warp], warp, lane, k); };
    auto row_of = [&](int b, int z) { return Ain + (long long)b * a_in_stride + (long long)z * pl.pitch; };

    // TM: a thread's 16 inputs per y task are the same in all four quarters: quarter 0 takes them from the landing zone and
    // parks them in tensor memory, the quarters 1..3 fetch them from there (no bulk copy, no landing-zone reads; the row of
    // A is read once per plane instead of four times).  !TM: a warp has more y tasks than its columns of tensor memory hold.
    __shared__ unsigned tm_slot;
    unsigned tm_warp = 0; // this warp's columns of tensor memory: lanes 32 (warp % 4) .., columns 256 (warp / 4) ..
    if (tid == 0) {
        for (int w = 0; w < NW; ++w) mbar_init(&bar_zone[w], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if constexpr (TM) {
        if (warp == 0) tmem_alloc(&tm_slot, 512);
        tmem_publish();
        tm_warp = tm_slot + ((unsigned)((warp & 3) * 32) << 16) + (unsigned)((warp >> 2) * 256);
    } else {
        __syncthreads();
    }
    int z = blockIdx.x % pl.n3, b = blockIdx.x / pl.n3;
    const int dz = gridDim.x % pl.n3, db = gridDim.x / pl.n3;
    if (kplanes > 0 && ytasks_w > 0) zone_issue(row_of(b, z), 0);

#pragma unroll 1
    for (int i = 0; i < kplanes; ++i) {
        const int zc = z + dz, zn = zc >= pl.n3 ? zc - pl.n3 : zc, bn = b + db + (zc >= pl.n3 ? 1 : 0); // next plane
        const bool more = i + 1 < kplanes;
        const C *row = row_of(b, z);
        // ================================================== Y_R: columns -> pbuf (lines y = 4 y' + R)
        auto yphase = [&](auto rc) {
            constexpr int R = decltype(rc)::value;
            C sv = czero<T>(); // single-stick column of this warp: its value, loaded while the y tasks run
            int4 sco = make_int4(0, 0, 0, 0);
            int scol = 0;
            if (warp < n_one) {
                scol = ct.perm[pl.n_multi + warp];
                sco = ct.col[scol];
                sv = __ldcg(row + sco.x);
            }
#pragma unroll 1
            for (int k = 0; k < ytasks_w; ++k) {
                const int4 d = ts.desc[warp][k][f]; // {first value in the zone, stick count, k2lo, column}
                const bool act = d.y > 0;
                const int ic = M - d.z;
                const bool hc = t == 0 && (unsigned)ic < (unsigned)d.y; // the +N/4 alias: one column at most
                C a[8], bq[8], u[8], y[1][8], cv;
                if constexpr (TM && R > 0) {
                    typename TmemWords<T>::type wds;
                    tmem_get16_issue(tm_warp + (unsigned)(k * tmem_cols16<T>()), wds);
                    cv = hc ? __ldcg(row + ts.copy[warp][k][f].w + ic) : czero<T>();
                    tmem_wait_ld();
                    tmem_unpack16(wds, a, bq);
                } else {
                    mbar_wait(&bar_zone[warp], zone_par);
                    zone_par ^= 1u;
                    const C *src = zone + d.x;
#pragma unroll
                    for (int j = 0; j < 8; ++j) {
                        const int ia = (t + 8 * j) - M - d.z, ib = (t + 8 * j) - d.z;
                        a[j] = ((unsigned)ia < (unsigned)d.y) ? src[ia] : czero<T>();
                        bq[j] = ((unsigned)ib < (unsigned)d.y) ? src[ib] : czero<T>();
                    }
                    cv = hc ? src[ic] : czero<T>();
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                    __syncwarp(); // every lane has its values: the landing zone may be refilled
                    if constexpr (TM) {
                        // the zone is used in quarter 0 only: the next task of this plane, or the first one of the next plane
                        // (the first task of the next plane is requested when this plane's x tasks have left the zone)
                        if (k + 1 < ytasks_w) zone_issue(row, k + 1);
                        tmem_put16(tm_warp + (unsigned)(k * tmem_cols16<T>()), a, bq);
                        tmem_wait_st();
                    } else {
                        // next y task of this warp: same quarter, next quarter (same row again), or the next plane
                        if (k + 1 < ytasks_w) zone_issue(row, k + 1);
                        else if (R < 3) zone_issue(row, 0);
                        else if (more) zone_issue(row_of(bn, zn), 0);
                    }
                }
                r4_fold_inv<R, 0, T>(a, bq, cv, u, wt[R]);
                C *pc = pbuf + d.w * YP;
                sub_inv<F, T>(u, y, tws, ExSkew<T, P2, 1>{pc, act}, t); // exchanged in place in the column
                __syncwarp();
                if (act) {
#pragma unroll
                    for (int q = 0; q < 8; ++q) pc[t + 8 * q] = y[0][q];
                }
            }
            if (warp < n_one) // closed form x W^{k2 y}
                for (int yl = lane; yl < M; yl += 32) pbuf[scol * YP + yl] = cmul(sv, tw[(sco.z * (4 * yl + R)) & (N - 1)]);
            for (int k = warp + NW; k < n_one; k += NW) { // more single-stick columns than warps (explicit maps)
                const int col = ct.perm[pl.n_multi + k];
                const int4 co = ct.col[col];
                const C xv = __ldcg(row + co.x);
                for (int yl = lane; yl < M; yl += 32) pbuf[col * YP + yl] = cmul(xv, tw[(co.z * (4 * yl + R)) & (N - 1)]);
            }
        };
        // ================================================== X_r: 64 lines y = 4 y' + r -> cuboid
        // (r is a run-time value: the x phase is most of the code and exists once -- with the four quarters
        // unrolled the kernel outgrows the instruction caches)
        // TM: the zone is a landing zone in quarter 0's y phase only, so the x tasks stage their results there -- one half
        // (e = 0, 1 or 2, 3) of the (x, x+1) pairs of the task's four lines, dense [line][n'][pair] -- and ONE tensor copy
        // scatters them into the cuboid (the tensor of plane_r4_fwd_k): the stores do not hold registers and do not go
        // through the 32 B/clk store port (0.598 -> 0.584 ms on config 5).  !TM: 32-byte stores from the registers.
        auto stage_out = [&](const C (&o0)[1][8], const C (&o1)[1][8], int half, int r, int ylg) {
            if (lane == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); // the previous box has left the zone
            __syncwarp();
            const bool sw = sizeof(C) == 16 && t >= 4; // see box_read of plane_r4_fwd_k
            C *st = zone + f * (2 * M);
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const int n = 2 * (t + 8 * q);
                st[n + (sw ? 1 : 0)] = sw ? o1[0][q] : o0[0][q];
                st[n + (sw ? 0 : 1)] = sw ? o0[0][q] : o1[0][q];
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncwarp();
            if (lane == 0) {
                r4_lines_box_store(&cmap, half, r, ylg, zone);
                asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            }
        };
        auto xphase = [&](int r) {
#pragma unroll 1
            for (int v = 0; v < XT; ++v) {
                const int yl = (warp + v * NW) * G + f;
                C a[8], bq[8];
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int ca = (t + 8 * j) - M - k1lo, cb = (t + 8 * j) - k1lo;
                    a[j] = (unsigned)ca < (unsigned)nx ? pbuf[ca * YP + yl] : czero<T>();
                    bq[j] = (unsigned)cb < (unsigned)nx ? pbuf[cb * YP + yl] : czero<T>();
                }
                const int cc = M - k1lo;
                const C cv = (t == 0 && (unsigned)cc < (unsigned)nx) ? pbuf[cc * YP + yl] : czero<T>();
                C *rowo = cub_out + (((long long)b * pl.n3 + z) * N + (4 * yl + r)) * N;
                const int ylg = ((b * pl.n3 + z) * M) + (warp + v * NW) * G; // the task's first line, in units of four rows
                const ExSkew<T, P2, YP> ex{pbuf + yl, true}; // the line's slots are dead: exchanged in them
                C u[8], o0[1][8], o1[1][8];
                r4_fold_inv<0, 0, T>(a, bq, cv, u, wt[0]);
                sub_inv<F, T>(u, o0, tws, ex, t);
                r4_fold_inv<1, 0, T>(a, bq, cv, u, wt[1]);
                sub_inv<F, T>(u, o1, tws, ex, t);
                if constexpr (TM) {
                    stage_out(o0, o1, 0, r, ylg);
                } else {
#pragma unroll
                    for (int q = 0; q < 8; ++q) st_pair(rowo + 4 * (t + 8 * q), o0[0][q], o1[0][q]);
                }
                r4_fold_inv<2, 0, T>(a, bq, cv, u, wt[2]);
                sub_inv<F, T>(u, o0, tws, ex, t);
                r4_fold_inv<3, 0, T>(a, bq, cv, u, wt[3]);
                sub_inv<F, T>(u, o1, tws, ex, t);
                if constexpr (TM) {
                    stage_out(o0, o1, 1, r, ylg);
                } else {
#pragma unroll
                    for (int q = 0; q < 8; ++q) st_pair(rowo + 4 * (t + 8 * q) + 2, o0[0][q], o1[0][q]);
                }
            }
        };
#pragma unroll 1
        for (int r = 0; r < 4; ++r) {
            switch (r) {
            case 0: yphase(std::integral_constant<int, 0>{}); break;
            case 1: yphase(std::integral_constant<int, 1>{}); break;
            case 2: yphase(std::integral_constant<int, 2>{}); break;
            default: yphase(std::integral_constant<int, 3>{}); break;
            }
            __syncthreads();
            xphase(r);
            __syncthreads();
        }
        if constexpr (TM) {
            // the last box of this plane has left the zone: it is a landing zone again
            if (more && ytasks_w > 0) {
                if (lane == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
                __syncwarp();
                zone_issue(row_of(bn, zn), 0);
            }
        }
        z = zn; b = bn;
    }
    if constexpr (TM) {
        if (lane == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); // the boxes have been written
        tmem_publish(); // every warp is done with its columns
        if (warp == 0) tmem_dealloc(tm_slot, 512);
    }
}

// adjoint of r4_fold_inv: accumulate F[k] = sum_e conj(W^{e k}) G_e[k mod 64] for k = s - 64 (fa), s (fb), +64 (fc)
template <int E, int J, typename T>
__device__ __forceinline__ void r4_fold_fwd(const cx<T> (&gq)[8], cx<T> (&fa)[8], cx<T> (&fb)[8], cx<T> &fc, cx<T> wte)
{
    if constexpr (J < 8) {
        cx<T> h = gq[J];
        if constexpr (E > 0) h = cmulc(mul_root<(E * J) % 32, 32, -1, T>(h), wte); // conj(W^{E (t + 8 J)}) G
        if constexpr (E == 0) {
            fa[J] = h;
            fb[J] = h;
            if constexpr (J == 0) fc = h;
        } else {
            fb[J] = cadd(fb[J], h);
            fa[J] = cadd(fa[J], mul_root<(8 * E) % 32, 32, +1, T>(h));            // conj((-j)^E) = (+j)^E
            if constexpr (J == 0) fc = cadd(fc, mul_root<(32 - 8 * E) % 32, 32, +1, T>(h)); // conj((+j)^E)
        }
        r4_fold_fwd<E, J + 1, T>(gq, fa, fb, fc, wte);
    }
}

// the part of residue R of F[k] (added into the one plane of A by plane_r4_fwd_k):
// conj(W^{R k}) G_R[k mod 64] for k = s - 64 (pa), s (pb), +64 (pc)
template <int R, int J, typename T>
__device__ __forceinline__ void r4_part_fwd(const cx<T> (&gq)[8], cx<T> (&pa)[8], cx<T> (&pb)[8], cx<T> &pc, cx<T> wte)
{
    if constexpr (J < 8) {
        cx<T> h = gq[J];
        if constexpr (R > 0) h = cmulc(mul_root<(R * J) % 32, 32, -1, T>(h), wte);
        pb[J] = h;
        pa[J] = mul_root<(8 * R) % 32, 32, +1, T>(h);
        if constexpr (J == 0) pc = mul_root<(32 - 8 * R) % 32, 32, +1, T>(h);
        r4_part_fwd<R, J + 1, T>(gq, pa, pb, pc, wte);
    }
}

// ---------------------------------------------------------------------------------------------
// forward plane kernel of the 256 pattern: the adjoint chain, quarter by quarter.
//     X_r: each of the 64 lines y = 4 y' + r: (x, x+1) pairs loaded in two batches (e = 0,1 and e = 2,3),
//          four length-64 transforms, F[k1] accumulated over e -> the occupied k1 columns of pbuf    | barrier
//     Y_r: every column: length-64 transform over y', the part of residue r of F[k2] is ADDED to the parts of the
//          residues before it; residue 3 stores the sum into the one plane A[b][z][.]                    | barrier
// Where the running sums live (TM): the same thread handles the same columns in every quarter, so it parks its 16 values
// per y task in TENSOR MEMORY (tcgen05.st / tcgen05.ld, fftb_tmem.cuh: 256 columns per warp, two warps per lane
// quarter) -- A is written once and never read.  !TM (a warp has more y tasks than its columns hold: complex128 maps
// with more than 128 multi-stick columns): read-modify-write of the plane of A through L2, as in round 1.  Measured on
// config 5: 0.833 -> 0.670 ms per launch, bit-identical results (the sums are formed in the same order).
// The quarter-plane buffer leaves no room for a landing zone of G = 4 whole lines (4 KB each) per warp, but a sub-transform
// pair e = 0, 1 (or 2, 3) needs only every other (x, x+1) pair of a line: the cuboid is described to the TMA engine as a
// 5-dimensional tensor (4 doubles | half | n' | y mod 4 | y / 4 over all planes and bands), and ONE tensor copy gathers a
// half of the pairs of a task's four lines -- 32-byte pieces 64 bytes apart -- into 8 KB of shared memory, dense
// [line][n'][pair].  The second half of a task lands while its first two transforms run, the first half of the next
// task during the last two: no warp waits for a register load any more (round 1-2: two batches of 32-byte loads into
// registers, `long_scoreboard` the kernel's largest stall; 0.659 -> 0.595 ms on config 5, bit-identical).
// ---------------------------------------------------------------------------------------------
template <typename T, int NW, bool TM>
__global__ void __launch_bounds__(NW * 32, 1)
plane_r4_fwd_k(const __grid_constant__ DevPlan pl, const __grid_constant__ ColTab4 ct, const __grid_constant__ CUtensorMap cmap,
               cx<T> *__restrict__ Aout, long long a_out_stride, int nplanes)
{
    using C = cx<T>;
    using R4 = PlaneR4<T, NW>;
    using F = typename R4::F;
    constexpr int N = R4::N, M = R4::M, P2 = F::P2, G = F::G, YP = R4::YP;
    constexpr int XT = R4::NXT / NW;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // the plane of A this kernel accumulates its four y residues into is read and rewritten within microseconds: keep it in L2
    const unsigned long long pol_keep = l2_policy(2);
    C *pbuf = reinterpret_cast<C *>(smem_raw);
    // landing zone of this warp: one half (e = 0, 1 or e = 2, 3) of the (x, x+1) pairs of the G lines of an x task, dense
    // [line][n'][pair]; a tensor copy's destination must be 128-byte aligned
    unsigned char *lz_raw = smem_raw + sizeof(C) * (size_t)R4::PB;
    lz_raw += (128u - (smem_u32(lz_raw) & 127u)) & 127u;
    C *lzone = reinterpret_cast<C *>(lz_raw) + (size_t)(threadIdx.x >> 5) * R4::LZE;
    __shared__ __align__(8) unsigned long long bar_lz[NW], bar_pb;
    unsigned lz_par = 0, pb_par = 0;
    bool pb_pending = false;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int f = lane / P2, t = lane % P2;
    const C *tw = reinterpret_cast<const C *>(pl.tw1);
    C tws[8];
#pragma unroll
    for (int m = 1; m < 8; ++m) tws[m] = tw[(4 * t * m) & (N - 1)];
    tws[0] = mk<T>((T)1, (T)0);
    C wt[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) wt[e] = tw[e * t];
    const int nx = pl.nxocc, k1lo = pl.k1lo;
    const int n_one = nx - pl.n_multi;
    const int ntask_y = ycol_tasks<F>(pl.n_multi);
    const int kplanes = nplanes > (int)blockIdx.x ? (nplanes - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;
    int z = blockIdx.x % pl.n3, b = blockIdx.x / pl.n3;
    const int dz = gridDim.x % pl.n3, db = gridDim.x / pl.n3;
    const int ytasks_w = ntask_y > warp ? (ntask_y - warp + NW - 1) / NW : 0; // y tasks of this warp per quarter
    __shared__ R4Tasks<T, NW> ts;
    __shared__ unsigned tm_slot;
    r4_tasks_rows<T, NW>(ts, pl, ct, warp, lane, ytasks_w);
    if (tid == 0) {
        for (int w = 0; w < NW; ++w) mbar_init(&bar_lz[w], 1);
        mbar_init(&bar_pb, NW * 32);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if constexpr (!TM) __syncthreads();
    unsigned tm_warp = 0; // this warp's columns of tensor memory: lanes 32 (warp % 4) .., columns 256 (warp / 4) ..
    if constexpr (TM) {
        if (warp == 0) tmem_alloc(&tm_slot, 512);
        tmem_publish();
        tm_warp = tm_slot + ((unsigned)((warp & 3) * 32) << 16) + (unsigned)((warp >> 2) * 256);
    }

    // split barrier in front of a quarter's x phase (see plane_pf_k): a warp arrives when it is done with the quarter's y phase
    // and waits only where its next x task first touches the plane buffer (0.595 -> 0.574 ms on config 5; the same split in
    // front of the inverse kernel's y phases gained nothing and is not there)
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
    // box of (plane (bb, zz), quarter rr, x task vv of this warp, half hh) -> this warp's landing zone
    auto box_issue = [&](int bb, int zz, int rr, int vv, int hh) {
        if (lane == 0) {
            mbar_expect_tx(&bar_lz[warp], (unsigned)(R4::LZE * sizeof(C)));
            r4_lines_box_load(lzone, &cmap, hh, rr, ((bb * pl.n3 + zz) * M) + (warp + vv * NW) * G, &bar_lz[warp]);
        }
    };
    // ... and from there into the registers: o0 = x = 4 n' + 2 h, o1 = x = 4 n' + 2 h + 1, n' = t + 8 q
    auto box_read = [&](C (&o0)[1][8], C (&o1)[1][8]) {
        mbar_wait(&bar_lz[warp], lz_par);
        lz_par ^= 1u;
        // 16-byte elements: half of the lanes take the odd element first, so that the 32-byte-strided 16-byte reads of a
        // quarter warp fall into different bank groups (8-byte elements: a pair is one 16-byte access)
        const bool sw = sizeof(C) == 16 && t >= 4;
        const C *st = lzone + f * (2 * M);
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const int n = 2 * (t + 8 * q);
            const C va = st[n + (sw ? 1 : 0)], vb = st[n + (sw ? 0 : 1)];
            o0[0][q].x = sw ? vb.x : va.x; o0[0][q].y = sw ? vb.y : va.y;
            o1[0][q].x = sw ? va.x : vb.x; o1[0][q].y = sw ? va.y : vb.y;
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp(); // every lane has its values: the landing zone may be refilled
    };
    if (kplanes > 0) box_issue(b, z, 0, 0, 0);

#pragma unroll 1
    for (int i = 0; i < kplanes; ++i) {
        const int zc = z + dz, zn = zc >= pl.n3 ? zc - pl.n3 : zc, bn = b + db + (zc >= pl.n3 ? 1 : 0); // next plane
        const bool more = i + 1 < kplanes;
        // ================================================== X_r: 64 lines y = 4 y' + r -> pbuf
        // (r is a run-time value: the x phase exists once, see plane_r4_inv_k)
        auto xphase = [&](int r) {
#pragma unroll 1
            for (int v = 0; v < XT; ++v) {
                const int yl = (warp + v * NW) * G + f;
                const ExSkew<T, P2, YP> ex{pbuf + yl, true}; // the line's slots are still unused: exchanged in them
                C o0[1][8], o1[1][8], gq[8], fa[8], fb[8], fc;
                box_read(o0, o1);
                box_issue(b, z, r, v, 1); // the other half of the same lines lands while e = 0, 1 are transformed
                sub_fwd_front<F, T>(o0, tws);
                sub_fwd_front<F, T>(o1, tws);
                pb_wait(); // the previous quarter's y phase is over in every warp
                sub_fwd_back<F, T>(o0, gq, ex, t);
                r4_fold_fwd<0, 0, T>(gq, fa, fb, fc, wt[0]);
                sub_fwd_back<F, T>(o1, gq, ex, t);
                r4_fold_fwd<1, 0, T>(gq, fa, fb, fc, wt[1]);
                box_read(o0, o1);
                // the first half of this warp's next x task: same quarter, next quarter, or the next plane
                if (v + 1 < XT) box_issue(b, z, r, v + 1, 0);
                else if (r < 3) box_issue(b, z, r + 1, 0, 0);
                else if (more) box_issue(bn, zn, 0, 0, 0);
                sub_fwd<F, T>(o0, gq, tws, ex, t);
                r4_fold_fwd<2, 0, T>(gq, fa, fb, fc, wt[2]);
                sub_fwd<F, T>(o1, gq, tws, ex, t);
                r4_fold_fwd<3, 0, T>(gq, fa, fb, fc, wt[3]);
                __syncwarp(); // the last exchange has been read by every lane: the slots take the results
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int ca = (t + 8 * j) - M - k1lo, cb = (t + 8 * j) - k1lo;
                    if ((unsigned)ca < (unsigned)nx) pbuf[ca * YP + yl] = fa[j];
                    if ((unsigned)cb < (unsigned)nx) pbuf[cb * YP + yl] = fb[j];
                }
                const int cc = M - k1lo;
                if (t == 0 && (unsigned)cc < (unsigned)nx) pbuf[cc * YP + yl] = fc;
            }
        };
        // ================================================== Y_R: columns -> partial plane R of A
        auto yphase = [&](auto rc) {
            constexpr int R = decltype(rc)::value;
            C *dst = Aout + (long long)b * a_out_stride + (long long)z * pl.pitch;
#pragma unroll 1
            for (int k = 0; k < ytasks_w; ++k) {
                const int4 co = ts.desc[warp][k][f]; // {first stick, stick count (0: no column), k2lo, column}
                const bool act = co.y > 0;
                C *pc = pbuf + co.w * YP;
                C *d = dst + co.x;
                const int ic = M - co.z;
                const bool hc = t == 0 && (unsigned)ic < (unsigned)co.y; // the +N/4 alias: one column at most, through L2
                C y[1][8], gq[8], pa[8], pb[8], pcv, oc = czero<T>();
                if constexpr (TM) {
                    const unsigned taddr = tm_warp + (unsigned)(k * tmem_cols16<T>());
                    typename TmemWords<T>::type old;
                    if constexpr (R > 0) {
                        tmem_get16_issue(taddr, old); // lands while the column is transformed
                        if (hc) oc = ld_hint(d + ic, pol_keep);
                    }
#pragma unroll
                    for (int q = 0; q < 8; ++q) y[0][q] = pc[t + 8 * q];
                    sub_fwd<F, T>(y, gq, tws, ExSkew<T, P2, 1>{pc, act}, t); // exchanged in place in the column
                    r4_part_fwd<R, 0, T>(gq, pa, pb, pcv, wt[R]);
                    if constexpr (R > 0) {
                        tmem_wait_ld();
                        tmem_add16(old, pa, pb);
                    }
                    if constexpr (R < 3) {
                        tmem_put16(taddr, pa, pb);
                        tmem_wait_st();
                        if (hc) st_hint(d + ic, R > 0 ? cadd(oc, pcv) : pcv, pol_keep);
                    } else {
#pragma unroll
                        for (int j = 0; j < 8; ++j) {
                            const int ia = (t + 8 * j) - M - co.z, ib = (t + 8 * j) - co.z;
                            if ((unsigned)ia < (unsigned)co.y) d[ia] = pa[j];
                            if ((unsigned)ib < (unsigned)co.y) d[ib] = pb[j];
                        }
                        if (hc) d[ic] = cadd(oc, pcv);
                    }
                } else {
                    // residue 0 stores, residues 1..3 add to what the SAME lane stored one quarter ago (still in L2; the loads
                    // are issued before the transform whose result they are added to)
                    C oa[8], ob[8];
                    if constexpr (R > 0) {
#pragma unroll
                        for (int j = 0; j < 8; ++j) {
                            const int ia = (t + 8 * j) - M - co.z, ib = (t + 8 * j) - co.z;
                            oa[j] = ((unsigned)ia < (unsigned)co.y) ? ld_hint(d + ia, pol_keep) : czero<T>();
                            ob[j] = ((unsigned)ib < (unsigned)co.y) ? ld_hint(d + ib, pol_keep) : czero<T>();
                        }
                        if (hc) oc = ld_hint(d + ic, pol_keep);
                    }
#pragma unroll
                    for (int q = 0; q < 8; ++q) y[0][q] = pc[t + 8 * q];
                    sub_fwd<F, T>(y, gq, tws, ExSkew<T, P2, 1>{pc, act}, t); // exchanged in place in the column
                    r4_part_fwd<R, 0, T>(gq, pa, pb, pcv, wt[R]);
#pragma unroll
                    for (int j = 0; j < 8; ++j) {
                        const int ia = (t + 8 * j) - M - co.z, ib = (t + 8 * j) - co.z;
                        if ((unsigned)ia < (unsigned)co.y) st_hint(d + ia, R > 0 ? cadd(oa[j], pa[j]) : pa[j], pol_keep);
                        if ((unsigned)ib < (unsigned)co.y) st_hint(d + ib, R > 0 ? cadd(ob[j], pb[j]) : pb[j], pol_keep);
                    }
                    if (hc) st_hint(d + ic, R > 0 ? cadd(oc, pcv) : pcv, pol_keep);
                }
            }
            // single-stick columns: one warp per column, dot product with conj(W^{k2 y}) over the quarter's lines
            for (int k = warp; k < n_one; k += NW) {
                const int col = ct.perm[pl.n_multi + k];
                const int4 co = ct.col[col];
                C acc = czero<T>();
                for (int yl = lane; yl < M; yl += 32) acc = cadd(acc, cmulc(pbuf[col * YP + yl], tw[(co.z * (4 * yl + R)) & (N - 1)]));
#pragma unroll
                for (int sft = 16; sft > 0; sft >>= 1) {
                    acc.x += __shfl_xor_sync(0xffffffffu, acc.x, sft);
                    acc.y += __shfl_xor_sync(0xffffffffu, acc.y, sft);
                }
                if (lane == 0) st_hint(dst + co.x, R > 0 ? cadd(ld_hint(dst + co.x, pol_keep), acc) : acc, pol_keep);
            }
        };
#pragma unroll 1
        for (int r = 0; r < 4; ++r) {
            xphase(r);
            __syncthreads();
            switch (r) {
            case 0: yphase(std::integral_constant<int, 0>{}); break;
            case 1: yphase(std::integral_constant<int, 1>{}); break;
            case 2: yphase(std::integral_constant<int, 2>{}); break;
            default: yphase(std::integral_constant<int, 3>{}); break;
            }
            pb_arrive(); // split: waited for inside the next quarter's first x task
        }
        z = zn; b = bn;
    }
    if constexpr (TM) {
        tmem_publish(); // every warp is done with its columns
        if (warp == 0) tmem_dealloc(tm_slot, 512);
    }
}

// ---------------------------------------------------------------------------------------------
// fused local-potential apply of the 256 pattern: per quarter r
//     Y_inv_r (as plane_r4_inv_k)                                                        | barrier
//     X_r: a line's 129 inputs -> e = 0, 1: two transforms, times V(r), two adjoint transforms, F[k1]
//          accumulated; the inputs are read AGAIN from the plane buffer for e = 2, 3 (they would not fit in
//          registers next to F), so the exchanges go through the warp's landing zone instead of the line's
//          slots; finally F[k1] replaces the line in the plane buffer                      | barrier
//     Y_fwd_r (as plane_r4_fwd_k: added into one plane of A), then the Y_inv of the next quarter on the
//          same columns by the same warp, no barrier in between.
// The cuboid is never written (I6').  The landing zone is scratch during X_r, so the first y task of
// a quarter is requested after X_{r-1} and lands during Y_fwd_{r-1}.
// ---------------------------------------------------------------------------------------------
template <typename T, int NW, bool TM>
__global__ void __launch_bounds__(NW * 32, 1)
plane_r4_vloc_k(const __grid_constant__ DevPlan pl, const __grid_constant__ ColTab4 ct, const cx<T> *__restrict__ Ain,
                cx<T> *__restrict__ Aout, const T *__restrict__ vloc, long long a_in_stride, long long a_out_stride, int nplanes)
{
    using C = cx<T>;
    using R4 = PlaneR4<T, NW>;
    using F = typename R4::F;
    constexpr int N = R4::N, M = R4::M, P2 = F::P2, G = F::G, YP = R4::YP, ZCOL = R4::ZCOL;
    constexpr int XT = R4::NXT / NW;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // the plane of A this kernel accumulates its four y residues into is read and rewritten within microseconds: keep it in L2
    const unsigned long long pol_keep = l2_policy(2);
    C *pbuf = reinterpret_cast<C *>(smem_raw);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int f = lane / P2, t = lane % P2;
    C *zone = pbuf + R4::PB + warp * R4::ZONE;
    __shared__ __align__(8) unsigned long long bar_zone[NW];
    unsigned zone_par = 0;
    const C *tw = reinterpret_cast<const C *>(pl.tw1);
    C tws[8];
#pragma unroll
    for (int m = 1; m < 8; ++m) tws[m] = tw[(4 * t * m) & (N - 1)];
    tws[0] = mk<T>((T)1, (T)0);
    C wt[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) wt[e] = tw[e * t];
    const int nx = pl.nxocc, k1lo = pl.k1lo;
    const int n_one = nx - pl.n_multi;
    const int ntask_y = ycol_tasks<F>(pl.n_multi);
    const int kplanes = nplanes > (int)blockIdx.x ? (nplanes - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x : 0;
    const int ytasks_w = ntask_y > warp ? (ntask_y - warp + NW - 1) / NW : 0;

    __shared__ R4Tasks<T, NW> ts; // y-task descriptors of the warps, built once
    r4_tasks_zone<T, NW>(ts, pl, ct, warp, lane, ytasks_w);
    auto zone_issue = [&](const C *row, int k) { r4_zone_issue<T, NW>(ts, row, zone, &bar_zone[warp], warp, lane, k); };
    auto row_of = [&](int b, int z) { return Ain + (long long)b * a_in_stride + (long long)z * pl.pitch; };
    // TM: the running sums of the forward y passes live in tensor memory, as in plane_r4_fwd_k
    __shared__ unsigned tm_slot;
    unsigned tm_warp = 0;

    if (tid == 0) {
        for (int w = 0; w < NW; ++w) mbar_init(&bar_zone[w], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if constexpr (TM) {
        if (warp == 0) tmem_alloc(&tm_slot, 512);
        tmem_publish();
        tm_warp = tm_slot + ((unsigned)((warp & 3) * 32) << 16) + (unsigned)((warp >> 2) * 256);
    } else {
        __syncthreads();
    }
    int z = blockIdx.x % pl.n3, b = blockIdx.x / pl.n3;
    const int dz = gridDim.x % pl.n3, db = gridDim.x / pl.n3;
    if (kplanes > 0 && ytasks_w > 0) zone_issue(row_of(b, z), 0);

#pragma unroll 1
    for (int i = 0; i < kplanes; ++i) {
        const int zc = z + dz, zn = zc >= pl.n3 ? zc - pl.n3 : zc, bn = b + db + (zc >= pl.n3 ? 1 : 0);
        const bool more = i + 1 < kplanes;
        const C *row = row_of(b, z);
        C *dst = Aout + (long long)b * a_out_stride + (long long)z * pl.pitch;
        // ================================================== Y_inv_R: columns -> pbuf
        auto yinv = [&](auto rc) {
            constexpr int R = decltype(rc)::value;
            C sv = czero<T>();
            int4 sco = make_int4(0, 0, 0, 0);
            int scol = 0;
            if (warp < n_one) {
                scol = ct.perm[pl.n_multi + warp];
                sco = ct.col[scol];
                sv = __ldcg(row + sco.x);
            }
#pragma unroll 1
            for (int k = 0; k < ytasks_w; ++k) {
                const int4 d = ts.desc[warp][k][f]; // {first value in the zone, stick count, k2lo, column}
                const bool act = d.y > 0;
                mbar_wait(&bar_zone[warp], zone_par);
                zone_par ^= 1u;
                const C *src = zone + d.x;
                C a[8], bq[8], u[8], y[1][8];
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int ia = (t + 8 * j) - M - d.z, ib = (t + 8 * j) - d.z;
                    a[j] = ((unsigned)ia < (unsigned)d.y) ? src[ia] : czero<T>();
                    bq[j] = ((unsigned)ib < (unsigned)d.y) ? src[ib] : czero<T>();
                }
                const int ic = M - d.z;
                const C cv = (t == 0 && (unsigned)ic < (unsigned)d.y) ? src[ic] : czero<T>();
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                __syncwarp();
                if (k + 1 < ytasks_w) zone_issue(row, k + 1); // within the y phase the zone is a landing zone only
                r4_fold_inv<R, 0, T>(a, bq, cv, u, wt[R]);
                C *pc = pbuf + d.w * YP;
                sub_inv<F, T>(u, y, tws, ExSkew<T, P2, 1>{pc, act}, t);
                __syncwarp();
                if (act) {
#pragma unroll
                    for (int q = 0; q < 8; ++q) pc[t + 8 * q] = y[0][q];
                }
            }
            if (warp < n_one)
                for (int yl = lane; yl < M; yl += 32) pbuf[scol * YP + yl] = cmul(sv, tw[(sco.z * (4 * yl + R)) & (N - 1)]);
            for (int k = warp + NW; k < n_one; k += NW) { // more single-stick columns than warps (explicit maps)
                const int col = ct.perm[pl.n_multi + k];
                const int4 co = ct.col[col];
                const C xv = __ldcg(row + co.x);
                for (int yl = lane; yl < M; yl += 32) pbuf[col * YP + yl] = cmul(xv, tw[(co.z * (4 * yl + R)) & (N - 1)]);
            }
        };
        // ================================================== X_r: inverse, V(r), forward, in place in pbuf
        // (r is a run-time value here: this is the bulk of the code and it exists once, see the note on the
        // instruction cache in DESIGN.md 6.4)
        auto xphase = [&](int r) {
#pragma unroll 1
            for (int v = 0; v < XT; ++v) {
                const int yl = (warp + v * NW) * G + f;
                const T *vrow = vloc + ((long long)z * N + (4 * yl + r)) * N;
                const ExSkew<T, P2, 1> ex{zone + f * ZCOL, true}; // the line must stay intact for the second read
                C fa[8], fb[8], fc;
                auto pass = [&](auto ec) {
                    constexpr int E0 = decltype(ec)::value; // this pass does e = E0, E0 + 1
                    T v0[8], v1[8];
#pragma unroll
                    for (int q = 0; q < 8; ++q) { // V at x = 4 n' + E0, + 1: one load per pair
                        const C vv = __ldg(reinterpret_cast<const C *>(vrow + 4 * (t + 8 * q) + E0));
                        v0[q] = vv.x;
                        v1[q] = vv.y;
                    }
                    C a[8], bq[8];
#pragma unroll
                    for (int j = 0; j < 8; ++j) {
                        const int ca = (t + 8 * j) - M - k1lo, cb = (t + 8 * j) - k1lo;
                        a[j] = (unsigned)ca < (unsigned)nx ? pbuf[ca * YP + yl] : czero<T>();
                        bq[j] = (unsigned)cb < (unsigned)nx ? pbuf[cb * YP + yl] : czero<T>();
                    }
                    const int cc = M - k1lo;
                    const C cv = (t == 0 && (unsigned)cc < (unsigned)nx) ? pbuf[cc * YP + yl] : czero<T>();
                    C u[8], o0[1][8], o1[1][8], gq[8];
                    r4_fold_inv<E0, 0, T>(a, bq, cv, u, wt[E0]);
                    sub_inv<F, T>(u, o0, tws, ex, t);
                    r4_fold_inv<E0 + 1, 0, T>(a, bq, cv, u, wt[E0 + 1]);
                    sub_inv<F, T>(u, o1, tws, ex, t);
#pragma unroll
                    for (int q = 0; q < 8; ++q) {
                        o0[0][q].x *= v0[q]; o0[0][q].y *= v0[q];
                        o1[0][q].x *= v1[q]; o1[0][q].y *= v1[q];
                    }
                    sub_fwd<F, T>(o0, gq, tws, ex, t);
                    r4_fold_fwd<E0, 0, T>(gq, fa, fb, fc, wt[E0]);
                    sub_fwd<F, T>(o1, gq, tws, ex, t);
                    r4_fold_fwd<E0 + 1, 0, T>(gq, fa, fb, fc, wt[E0 + 1]);
                };
                pass(std::integral_constant<int, 0>{});
                pass(std::integral_constant<int, 2>{});
                __syncwarp(); // every lane has read the line twice: it takes the result
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int ca = (t + 8 * j) - M - k1lo, cb = (t + 8 * j) - k1lo;
                    if ((unsigned)ca < (unsigned)nx) pbuf[ca * YP + yl] = fa[j];
                    if ((unsigned)cb < (unsigned)nx) pbuf[cb * YP + yl] = fb[j];
                }
                const int cc = M - k1lo;
                if (t == 0 && (unsigned)cc < (unsigned)nx) pbuf[cc * YP + yl] = fc;
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); // generic-proxy writes to the zone before the next bulk copy
        };
        // ================================================== Y_fwd_R: columns -> added into the one plane of A
        auto yfwd = [&](auto rc) {
            constexpr int R = decltype(rc)::value;
#pragma unroll 1
            for (int k = 0; k < ytasks_w; ++k) {
                const int4 dk = ts.desc[warp][k][f]; // {., stick count (0: no column), k2lo, column}
                const int4 co = make_int4(ts.copy[warp][k][f].w, dk.y, dk.z, dk.w); // .x = first stick of the column in the row of A
                const bool act = co.y > 0;
                C *pc = pbuf + co.w * YP;
                C *d = dst + co.x;
                const int ic = M - co.z;
                const bool hc = t == 0 && (unsigned)ic < (unsigned)co.y; // the +N/4 alias: one column at most, through L2
                C y[1][8], gq[8], pa[8], pb[8], pcv, oc = czero<T>();
                if constexpr (TM) {
                    const unsigned taddr = tm_warp + (unsigned)(k * tmem_cols16<T>());
                    typename TmemWords<T>::type old;
                    if constexpr (R > 0) {
                        tmem_get16_issue(taddr, old); // lands while the column is transformed
                        if (hc) oc = ld_hint(d + ic, pol_keep);
                    }
#pragma unroll
                    for (int q = 0; q < 8; ++q) y[0][q] = pc[t + 8 * q];
                    sub_fwd<F, T>(y, gq, tws, ExSkew<T, P2, 1>{pc, act}, t);
                    r4_part_fwd<R, 0, T>(gq, pa, pb, pcv, wt[R]);
                    if constexpr (R > 0) {
                        tmem_wait_ld();
                        tmem_add16(old, pa, pb);
                    }
                    if constexpr (R < 3) {
                        tmem_put16(taddr, pa, pb);
                        tmem_wait_st();
                        if (hc) st_hint(d + ic, R > 0 ? cadd(oc, pcv) : pcv, pol_keep);
                    } else {
#pragma unroll
                        for (int j = 0; j < 8; ++j) {
                            const int ia = (t + 8 * j) - M - co.z, ib = (t + 8 * j) - co.z;
                            if ((unsigned)ia < (unsigned)co.y) d[ia] = pa[j];
                            if ((unsigned)ib < (unsigned)co.y) d[ib] = pb[j];
                        }
                        if (hc) d[ic] = cadd(oc, pcv);
                    }
                } else {
                    C oa[8], ob[8];
                    if constexpr (R > 0) {
#pragma unroll
                        for (int j = 0; j < 8; ++j) {
                            const int ia = (t + 8 * j) - M - co.z, ib = (t + 8 * j) - co.z;
                            oa[j] = ((unsigned)ia < (unsigned)co.y) ? ld_hint(d + ia, pol_keep) : czero<T>();
                            ob[j] = ((unsigned)ib < (unsigned)co.y) ? ld_hint(d + ib, pol_keep) : czero<T>();
                        }
                        if (hc) oc = ld_hint(d + ic, pol_keep);
                    }
#pragma unroll
                    for (int q = 0; q < 8; ++q) y[0][q] = pc[t + 8 * q];
                    sub_fwd<F, T>(y, gq, tws, ExSkew<T, P2, 1>{pc, act}, t);
                    r4_part_fwd<R, 0, T>(gq, pa, pb, pcv, wt[R]);
#pragma unroll
                    for (int j = 0; j < 8; ++j) {
                        const int ia = (t + 8 * j) - M - co.z, ib = (t + 8 * j) - co.z;
                        if ((unsigned)ia < (unsigned)co.y) st_hint(d + ia, R > 0 ? cadd(oa[j], pa[j]) : pa[j], pol_keep);
                        if ((unsigned)ib < (unsigned)co.y) st_hint(d + ib, R > 0 ? cadd(ob[j], pb[j]) : pb[j], pol_keep);
                    }
                    if (hc) st_hint(d + ic, R > 0 ? cadd(oc, pcv) : pcv, pol_keep);
                }
            }
            for (int k = warp; k < n_one; k += NW) {
                const int col = ct.perm[pl.n_multi + k];
                const int4 co = ct.col[col];
                C acc = czero<T>();
                for (int yl = lane; yl < M; yl += 32) acc = cadd(acc, cmulc(pbuf[col * YP + yl], tw[(co.z * (4 * yl + R)) & (N - 1)]));
#pragma unroll
                for (int sft = 16; sft > 0; sft >>= 1) {
                    acc.x += __shfl_xor_sync(0xffffffffu, acc.x, sft);
                    acc.y += __shfl_xor_sync(0xffffffffu, acc.y, sft);
                }
                if (lane == 0) st_hint(dst + co.x, R > 0 ? cadd(ld_hint(dst + co.x, pol_keep), acc) : acc, pol_keep);
            }
        };
        using I0 = std::integral_constant<int, 0>; using I1 = std::integral_constant<int, 1>;
        using I2 = std::integral_constant<int, 2>; using I3 = std::integral_constant<int, 3>;
#pragma unroll 1
        for (int r = 0; r < 4; ++r) {
            switch (r) {
            case 0: yinv(I0{}); break;
            case 1: yinv(I1{}); break;
            case 2: yinv(I2{}); break;
            default: yinv(I3{}); break;
            }
            __syncthreads();
            xphase(r);
            __syncthreads();
            // the zone is a landing zone again: the first y task of the next quarter (or plane) lands during Y_fwd_r
            if (ytasks_w > 0) {
                if (r < 3) zone_issue(row, 0);
                else if (more) zone_issue(row_of(bn, zn), 0);
            }
            switch (r) {
            case 0: yfwd(I0{}); break;
            case 1: yfwd(I1{}); break;
            case 2: yfwd(I2{}); break;
            default: yfwd(I3{}); break;
            }
            // no barrier: the next Y_inv touches the same columns from the same warp
        }
        z = zn; b = bn;
    }
    if constexpr (TM) {
        tmem_publish(); // every warp is done with its columns
        if (warp == 0) tmem_dealloc(tm_slot, 512);
    }
}

// ---------------------------------------------------------------------------------------------
// forward z pass of the 256 pattern for plans whose forward plane kernel writes partial planes of A (ry > 1: generic
// x/y patterns next to a 256 z axis), which it sums while it fills the tile: one group of 8 lanes per stick, TS = 4 NW
// sticks per CTA, the same tile transposition as zpass_fast_fwd_k (element (z, sl) in column (sl + z/4) mod TS: the
// strided accesses z = 4 n' + e of the transforms are conflict-free).  The inverse z pass and the forward one with a
// single plane of A are the persistent kernels of fftb_zpass_pf.cuh.
//   grid = (ceil(n_sticks / TS), bands)
// ---------------------------------------------------------------------------------------------
template <typename T, int NW> struct ZR4 {
    using F = FastCfg<T, 128, 8, 8>;
    static constexpr int N = 256, M = 64, TS = F::G * NW;
    static constexpr size_t smem_bytes = sizeof(cx<T>) * ((size_t)N * TS + (size_t)NW * F::EXW);
    static constexpr int GW = F::LW / F::P2 < 1 ? 1 : F::LW / F::P2; // lane groups per wavefront, see ZFast
    static_assert(TS >= F::LW, "tile row shorter than a wavefront");
    __device__ static __forceinline__ int rot(int z) { return (z >> 2) * GW; }
    __device__ static __forceinline__ int swz(int z, int sl) { return z * TS + ((sl + rot(z)) & (TS - 1)); }
};

template <typename T, int NW>
__global__ void __launch_bounds__(NW * 32, 2)
zpass_r4_fwd_k(const __grid_constant__ DevPlan pl, const cx<T> *__restrict__ A, cx<T> *__restrict__ packed, long long a_band_stride)
{
    using C = cx<T>;
    using Z = ZR4<T, NW>;
    using F = typename Z::F;
    constexpr int N = Z::N, M = Z::M, P2 = F::P2, G = F::G, TS = Z::TS, NT = NW * 32;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C *tile = reinterpret_cast<C *>(smem_raw);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int f = lane / P2, t = lane % P2;
    const ExTile<T, P2> ex{tile + N * TS + warp * F::EXW + f * F::FS};
    const C *tw = reinterpret_cast<const C *>(pl.tw3);
    const int s0 = blockIdx.x * TS, sl = warp * G + f, s = s0 + sl;
    const bool act = s < pl.nsticks;
    // ---- A[z][s0 .. s0+TS) -> tile, summing the ry partial planes of the forward plane kernel
    {
        const C *src = A + (long long)blockIdx.y * a_band_stride + s0;
        const long long rstride = (long long)pl.n3 * pl.pitch;
        constexpr int U = 8;
        static_assert((N * TS) % (NT * U) == 0, "tile copy is unrolled by U");
        for (int i0 = tid; i0 < N * TS; i0 += NT * U) {
            C v[U];
#pragma unroll
            for (int uu = 0; uu < U; ++uu) {
                const int i = i0 + uu * NT, z = i / TS, l = i % TS;
                v[uu] = (s0 + l < pl.nsticks) ? __ldcg(src + (long long)z * pl.pitch + l) : czero<T>();
            }
            for (int p = 1; p < pl.ry; ++p) {
#pragma unroll
                for (int uu = 0; uu < U; ++uu) {
                    const int i = i0 + uu * NT, z = i / TS, l = i % TS;
                    if (s0 + l < pl.nsticks) v[uu] = cadd(v[uu], __ldcg(src + p * rstride + (long long)z * pl.pitch + l));
                }
            }
#pragma unroll
            for (int uu = 0; uu < U; ++uu) {
                const int i = i0 + uu * NT, z = i / TS, l = i % TS;
                tile[Z::swz(z, l)] = v[uu];
            }
        }
    }
    C tws[8], wt[4];
#pragma unroll
    for (int m = 1; m < 8; ++m) tws[m] = tw[(4 * t * m) & (N - 1)];
    tws[0] = mk<T>((T)1, (T)0);
#pragma unroll
    for (int e = 0; e < 4; ++e) wt[e] = tw[e * t];
    const int4 st = pl.stick[act ? s : 0];
    C *dst = packed + (long long)blockIdx.y * pl.S + st.x;
    const T scale = (T)pl.scale;
    __syncthreads();
    C y[1][8], gq[8], fa[8], fb[8], fc;
#pragma unroll
    for (int q = 0; q < 8; ++q) y[0][q] = tile[Z::swz(4 * (t + 8 * q), sl)];
    sub_fwd<F, T>(y, gq, tws, ex, t);
    r4_fold_fwd<0, 0, T>(gq, fa, fb, fc, wt[0]);
#pragma unroll
    for (int q = 0; q < 8; ++q) y[0][q] = tile[Z::swz(4 * (t + 8 * q) + 1, sl)];
    sub_fwd<F, T>(y, gq, tws, ex, t);
    r4_fold_fwd<1, 0, T>(gq, fa, fb, fc, wt[1]);
#pragma unroll
    for (int q = 0; q < 8; ++q) y[0][q] = tile[Z::swz(4 * (t + 8 * q) + 2, sl)];
    sub_fwd<F, T>(y, gq, tws, ex, t);
    r4_fold_fwd<2, 0, T>(gq, fa, fb, fc, wt[2]);
#pragma unroll
    for (int q = 0; q < 8; ++q) y[0][q] = tile[Z::swz(4 * (t + 8 * q) + 3, sl)];
    sub_fwd<F, T>(y, gq, tws, ex, t);
    r4_fold_fwd<3, 0, T>(gq, fa, fb, fc, wt[3]);
    if (act) {
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const int ia = (t + 8 * j) - M - st.y, ib = (t + 8 * j) - st.y;
            if ((unsigned)ia < (unsigned)st.z) dst[ia] = mk<T>(fa[j].x * scale, fa[j].y * scale);
            if ((unsigned)ib < (unsigned)st.z) dst[ib] = mk<T>(fb[j].x * scale, fb[j].y * scale);
        }
        const int ic = M - st.y;
        if (t == 0 && (unsigned)ic < (unsigned)st.z) dst[ic] = mk<T>(fc.x * scale, fc.y * scale);
    }
}

} // namespace fftb
