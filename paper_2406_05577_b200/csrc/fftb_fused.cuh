// fftb_fused.cuh -- one persistent launch per direction: z tiles AND z-planes of the whole batch (sm_100a).
//
// The separate z-pass and plane launches send the plane-major intermediate A[b][z][stick] through HBM twice per
// direction (27% of the DRAM bytes of a step, "keeping the amount of data moved ... to a minimum").
// Here both kinds of work item live in ONE cooperative launch, and A is a RING of `nslot` band slots (a few tens of
// MB) that is written and read in L2 and overwritten before it is ever evicted:
//
//   inverse   Z(b, j)  tile j of band b:  packed range -> pruned z-DFT -> rows of ring[b % nslot]        (I1-I3)
//             P(b, z)  plane z of band b: row of ring[b % nslot] -> y-DFT, x-DFT -> cuboid             (I4-I7)
//   forward   P(b, z)  cuboid plane -> x-DFT, y-DFT -> row of ring[b % nslot]                           (F1-F4)
//             Z(b, j)  rows of ring[b % nslot] -> z-DFT, scale -> packed range                          (F5-F6)
//
// Items are dealt round-robin over the CTAs (tile w = b ntiles + j to CTA w mod G, plane p = b n3 + z to CTA
// p mod G), and every CTA walks its two lists merged by a KEY: inverse key(Z(b)) = b - lead - 1/2, key(P(b)) = b;
// forward key(P(b)) = b, key(Z(b)) = b + lead + 1/2.  Dependencies go through per-band counters in global memory:
//   inverse   P(b, .) needs zdone[b] == ntiles;  Z(b, .) may overwrite its slot once pdone[b - nslot] == n3
//   forward   Z(b, .) needs pdone[b] == n3;      P(b, .) may overwrite its slot once zdone[b - nslot] == ntiles
// Every dependency points to a smaller key (nslot > lead), every CTA is resident (cooperative launch) and works in
// key order, and a CTA publishes everything it has finished before it blocks: the unfinished item with the globally
// smallest key can always run, so the schedule cannot deadlock.  With lead >= 2 bands the producers run far enough
// ahead that a consumer practically never waits.
// Variant (kernel argument nz > 0, fftb_plan_tuning.z_ctas): a SPATIAL split -- CTAs 0 .. nz-1 walk the z tiles only,
// the others the planes only, each list still in band order, so the same argument holds; the z CTAs then run as far
// ahead as the ring allows (nslot bands) and `lead` plays no part.
//
// Ring layout.  The TMA engine of an SM takes a bulk copy about every 19 cycles (measured), so a z tile that leaves as
// one copy per z row (128 of them) would keep the CTA waiting for 2 500 cycles.  A ring slot is therefore TILE-MAJOR:
//     slot = [ntiles][the shared-memory image of a tile: ZFast::TILE elements, row z of the tile at ZFast::lin(z, 0)]
// A z tile leaves (inverse) or arrives (forward) as ONE contiguous bulk copy; the row of plane z -- TS elements out of
// every tile -- arrives in the inverse plane item as ONE 5-dimensional tensor copy (cp.async.bulk.tensor through a
// CUtensorMap over the ring: TS x parity x z pair x tile x slot, box = TS x 1 x 1 x ntiles x 1), which lands in stick
// order; the forward plane item writes its row with plain stores at the same addresses.
//
// The work inside an item is the code of fftb_plane_pf.cuh (plane) and fftb_zpass_pf.cuh (z tile, here with all NW
// warps of the CTA on one tile of G NW sticks).  The input of the NEXT item, whatever its kind, is requested from
// the TMA engine while the current one is transformed; the z tile shares the shared memory of the plane buffers.
#pragma once
#include "fftb_zpass_pf.cuh"
#include <cuda.h>

namespace fftb {

// Counters in global memory order the items of different CTAs.  A consumer polls with RELAXED loads and lets a
// control dependency order what follows: everything it then does with the data is a TMA bulk copy or a store that
// cannot be issued before the load has returned, and the data itself is read from L2, where the producer's release
// (or the completion of its bulk stores) put it before the counter moved.  An acquire load would cost an L1
// invalidation and well over a thousand cycles per item (measured), on the one thread every CTA barrier waits for.
__device__ __forceinline__ int ld_relaxed_gpu(const int *p)
{
    int v;
    asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void red_release_gpu(int *p)
{
    asm volatile("red.release.gpu.global.add.s32 [%0], 1;" ::"l"(p) : "memory");
}
__device__ __forceinline__ void red_relaxed_gpu(int *p)
{
    asm volatile("red.relaxed.gpu.global.add.s32 [%0], 1;" ::"l"(p) : "memory");
}
__device__ __forceinline__ void spin_until_ge(const int *p, int target)
{
    while (ld_relaxed_gpu(p) < target) __nanosleep(32);
}
__device__ __forceinline__ void bulk_load_hint(void *sdst, const void *gsrc, unsigned bytes, unsigned long long *bar, unsigned long long pol)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(smem_u32(sdst)),
                 "l"(gsrc), "r"(bytes), "r"(smem_u32(bar)), "l"(pol)
                 : "memory");
}
// row of plane z (coordinates: parity, z pair, slot) out of every tile of a ring slot; see the layout above
__device__ __forceinline__ void ring_row_load(void *sdst, const void *tmap, int parity, int zpair, int slot, unsigned long long *bar,
                                              unsigned long long pol)
{
    asm volatile("cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3, %4, %5, %6}], [%7], %8;" ::"r"(smem_u32(sdst)),
                 "l"(tmap), "r"(0), "r"(parity), "r"(zpair), "r"(0), "r"(slot), "r"(smem_u32(bar)), "l"(pol)
                 : "memory");
}
__device__ __forceinline__ void bulk_store_hint(void *gdst, const void *ssrc, unsigned bytes, unsigned long long pol)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;" ::"l"(gdst),
                 "r"((unsigned)__cvta_generic_to_shared(ssrc)), "r"(bytes), "l"(pol)
                 : "memory");
}
constexpr int fused_max(int a, int b) { return a > b ? a : b; }
constexpr int fused_even(int x) { return (x + 1) & ~1; }

template <typename T, class F, int NW> struct Fused {
    using PF = PlanePF<T, F, NW>;
    using Z = ZFast<T, F, NW>;
    using ZP = ZPers<T, F, NW>;
    // inverse: region P = the two plane buffers | z tile + the warps' exchange tiles; then the landing zone (row of A | packed range)
    static constexpr int A128 = 128 / (int)sizeof(cx<T>); // elements per 128 bytes: the tensor copy's destination alignment
    static constexpr int REGP_INV = (fused_max(2 * PF::PB, Z::TILE + NW * F::EXW) + A128 - 1) / A128 * A128;
    // forward: region P = the two plane buffers | exchange tiles + packed results; region L = cuboid lines of the warps | z tile
    static constexpr int REGP_FWD = fused_even(fused_max(2 * PF::PB, NW * F::EXW + ZP::LZ));
    static constexpr int REGL_FWD = fused_even(fused_max(NW * F::G * F::N, Z::TILE));
    // landing zone of the inverse kernel: a plane's row out of every tile (ntiles x TS elements) or a tile's packed range
    static size_t smem_inv(int ntiles)
    {
        const int land = ntiles * Z::TS > ZP::LZ ? ntiles * Z::TS : ZP::LZ;
        return sizeof(cx<T>) * ((size_t)REGP_INV + (size_t)fused_even(land)) + 128; // + alignment slack
    }
    static constexpr size_t smem_fwd = sizeof(cx<T>) * ((size_t)REGP_FWD + (size_t)REGL_FWD);
};

// =====================================================================================================================
// inverse
// =====================================================================================================================
template <typename T, class F, int NW>
__global__ void __launch_bounds__(NW * 32, 1)
fused_inv_k(const __grid_constant__ DevPlan pl, const __grid_constant__ ColTab ct, const cx<T> *__restrict__ packed,
            cx<T> *__restrict__ ring, const __grid_constant__ CUtensorMap ring_map, cx<T> *__restrict__ cub_out, long long slot_stride,
            int nb, int nslot, int lead, int nz, int hints, int *__restrict__ zdone, int *__restrict__ pdone)
{
    using C = cx<T>;
    using FU = Fused<T, F, NW>;
    using PF = typename FU::PF;
    using Z = typename FU::Z;
    constexpr int N = F::N, M = F::M, P1 = F::P1, P2 = F::P2, B2 = F::B2, G = F::G, YP = F::YP;
    constexpr int PB = PF::PB, XT = PF::XT, TS = Z::TS;
    constexpr long long EA = FU::ZP::EA;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // the tensor copy's destination (the landing zone) must be 128-byte aligned: the kernel gets 128 bytes of slack
    unsigned char *const smem_al = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
    C *const pb0 = reinterpret_cast<C *>(smem_al), *const pb1 = pb0 + PB; // plane item: [2 residues][NCOL][YP]
    C *const tile = pb0;                                                    // z item: [N/2][RP] (Z::lin), then the exchange tiles
    C *const stage = pb0 + FU::REGP_INV;                                    // landing zone of the next item's input
    __shared__ __align__(8) unsigned long long bar_full;
    __shared__ int s_issued;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int f = lane / P2, t = lane % P2;
    const ExTile<T, P2> zex{tile + Z::TILE + warp * F::EXW + f * F::FS};
    const int sl = warp * G + f;
    const C *tw = reinterpret_cast<const C *>(pl.tw1); // N1 == N2 == N3: one table
    C tws[P1];
#pragma unroll
    for (int m = 1; m < P1; ++m) tws[m] = tw[modn<N>(2 * t * m)];
    tws[0] = mk<T>((T)1, (T)0);
    const C g = tw[t];
    const int nx = pl.nxocc, k1lo = pl.k1lo, n3 = pl.n3;
    const bool l0 = (t == 0);
    const int n_one = nx - pl.n_multi;
    const int ntask_y = ycol_tasks<F>(pl.n_multi);
    // `packed` may be only 8-byte aligned (complex64): indices count elements from the 16-byte boundary pk at or below it
    const long long mis = (long long)(((unsigned long long)packed / sizeof(C)) & (unsigned long long)(EA - 1));
    const C *pk = packed - mis;
    const long long nall = mis + (long long)nb * pl.S;

    const int ntiles = (pl.nsticks + TS - 1) / TS;
    const unsigned stage_bytes = (unsigned)(ntiles * TS) * (unsigned)sizeof(C); // a plane's row: TS elements of every tile

    // ---- plane item: column groups of the y pass (see plane_pf_k) -----------------------------------------------
    struct YCol { bool act; int col; int4 co; };
    auto ycol = [&](int task) -> YCol {
        YCol c;
        const int ci = ycol_index<F>(task, f);
        c.act = task < ntask_y && ci < pl.n_multi;
        c.col = ct.perm[c.act ? ci : 0];
        c.co = ct.col[c.col];
        return c;
    };
    const YCol yc0 = ycol(warp), yc1 = ycol(warp + NW);
    auto ycol_of = [&](int task) -> YCol { return task == warp ? yc0 : task == warp + NW ? yc1 : ycol(task); };
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
        sub_inv<F, T>(xs, y, tws, ExSkew<T, P2, 1>{pc, c.act}, t);
        __syncwarp();
        if (c.act) {
#pragma unroll
            for (int bb = 0; bb < B2; ++bb)
#pragma unroll
                for (int q = 0; q < P2; ++q) pc[(t + P2 * bb) + P1 * q] = y[bb][q];
        }
        x[P1 / 2] = csub(x[P1 / 2], bv);
        pre_inv<F, 0, T>(x, g);
        pc = pb1 + c.col * YP;
        sub_inv<F, T>(x, y, tws, ExSkew<T, P2, 1>{pc, c.act}, t);
        __syncwarp();
        if (c.act) {
#pragma unroll
            for (int bb = 0; bb < B2; ++bb)
#pragma unroll
                for (int q = 0; q < P2; ++q) pc[(t + P2 * bb) + P1 * q] = y[bb][q];
        }
    };
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
        sub_inv<F, T>(xs, o0, tws, ExSkew<T, P2, YP>{pbuf + yl, true}, t);
        x[P1 / 2] = csub(x[P1 / 2], bv);
        pre_inv<F, 0, T>(x, g);
        sub_inv<F, T>(x, o1, tws, ExSkew<T, P2, YP>{pbuf + yl, true}, t);
    };
    auto yinv_single = [&]() {
        for (int i = warp; i < n_one; i += NW) {
            const int col = ct.perm[pl.n_multi + i];
            const int4 co = ct.col[col];
            const C v = stage[co.x];
            for (int y = lane; y < N; y += 32) (y & 1 ? pb1 : pb0)[col * YP + (y >> 1)] = cmul(v, tw[modn<N>(co.z * y)]);
        }
    };

    // ---- z item: descriptor of a tile, loaded one item ahead and not touched before it is needed (the stick table
    // is in global memory; see zpass_pers_inv_k) --------------------------------------------------------------------
    struct ZD { int4 st; int x0, x1, band, s0; bool act; };
    auto describe = [&](int band, int j) -> ZD {
        ZD d;
        d.band = band, d.s0 = j * TS;
        const int s = d.s0 + sl, s1 = d.s0 + TS;
        d.act = s < pl.nsticks;
        d.st = pl.stick[d.act ? s : d.s0];
        d.x0 = pl.stick[d.s0].x;
        d.x1 = s1 < pl.nsticks ? pl.stick[s1].x : (int)pl.S;
        return d;
    };
    // packed range of the tile in elements of the whole batch, widened to 16-byte boundaries [a0, a1)
    auto range_of = [&](const ZD &d, long long &a0, long long &a1) {
        const long long g0 = (mis + (long long)d.band * pl.S) + d.x0, g1 = (mis + (long long)d.band * pl.S) + d.x1;
        a0 = g0 & ~(EA - 1);
        a1 = (g1 + EA - 1) & ~(EA - 1);
        if (a1 > nall) a1 = nall & ~(EA - 1);
    };
    const unsigned long long pol_ring = l2_policy(hints ? 2 : 0), pol_stream = l2_policy(hints ? 1 : 0);
    // thread 0: request the input of an item.  A plane's row exists once every z tile of its band is in the ring
    // (dep = the counter's value, read earlier); returns 0 without a request if that is not so yet.
    auto issue_input = [&](int kind, int b, int z, const ZD &zd, int dep) -> int {
        if (kind == 2) {
            if (dep < ntiles) return 0;
            mbar_expect_tx(&bar_full, stage_bytes);
            ring_row_load(stage, &ring_map, z & 1, z >> 1, b % nslot, &bar_full, pol_ring);
        } else {
            long long a0, a1;
            range_of(zd, a0, a1);
            const unsigned bytes = (unsigned)((a1 - a0) * (long long)sizeof(C));
            mbar_expect_tx(&bar_full, bytes);
            if (bytes) bulk_load_hint(stage, pk + a0, bytes, &bar_full, pol_stream);
        }
        return 1;
    };
    // thread 0, after its cp.async.bulk.wait_group 0: the finished z tile is complete in the ring (the bulk store has
    // written it to L2, which is where the consumers' TMA copies read it, before the counter moves; a release fence
    // here would wait for every cuboid store the SM still has in flight: 1 000 - 2 500 cycles, measured)
    auto publish_z = [&](int band) { red_relaxed_gpu(zdone + band); };

    // this CTA's next tile (band zb, tile zj) and next plane (band pb, plane pz); both lists advance by GD items
    // nz > 0 (spatial split): the first nz CTAs take the z tiles only, the others the planes only
    const int GD = (int)gridDim.x, bid = (int)blockIdx.x;
    const bool zrole = nz > 0 && bid < nz, prole = nz > 0 && bid >= nz;
    const int zs = nz > 0 ? nz : GD, pi = prole ? bid - nz : bid, ps = nz > 0 ? GD - nz : GD;
    int zb = prole ? nb : bid / ntiles, zj = bid % ntiles, pb = zrole ? nb : pi / n3, pz = pi % n3;
    const int dzb = zs / ntiles, dzj = zs % ntiles, dpb = ps / n3, dpz = ps % n3;
    bool run_z = false;
    auto peek = [&]() -> int { // 0 none, 1 z tile, 2 plane
        const bool hz = zb < nb, hp = pb < nb;
        if (!hz) return hp ? 2 : 0;
        if (!hp) return 1;
        // z tiles come in runs (one band more of lead once a run has started, if the ring has room for it: nslot must
        // exceed the largest lead): fewer switches between the two kinds of item
        return zb - lead - (run_z && nslot > lead + 1 ? 1 : 0) <= pb ? 1 : 2;
    };
    int kind = peek();
    // zc always describes this CTA's next z tile; it is reloaded when that tile's item starts, i.e. at least one item
    // before the values are looked at (no instruction waits for the table loads)
    ZD zc = describe(zb < nb ? zb : 0, zb < nb ? zj : 0);
    if (tid == 0) {
        mbar_init(&bar_full, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        s_issued = 1;
    }
    __syncthreads();
    if (tid == 0 && kind == 1) issue_input(1, 0, 0, zc, 0);
    ZD cur = zc;
    unsigned par = 0;
    int pend_z = -1;     // band of the last z tile whose completion has not been published yet
    bool prev_z = false; // the previous item was a z tile: the TMA engine may still be reading it from region P
    bool issued = kind == 1; // the input of the current item has been requested
#pragma unroll 1
    while (kind) {
        // the current item, then the next one
        const int cb = kind == 1 ? zb : pb, cz = pz;
        if (kind == 1) {
            cur = zc;
            zj += dzj; zb += dzb; if (zj >= ntiles) { zj -= ntiles; ++zb; }
            zc = describe(zb < nb ? zb : 0, zb < nb ? zj : 0);
        } else { pz += dpz; pb += dpb; if (pz >= n3) { pz -= n3; ++pb; } }
        run_z = kind == 1;
        const int nkind = peek();
        // counters this item will look at, read now (thread 0) so that their latency is hidden: the next plane's band
        // and, for a z tile, the previous user of its ring slot
        int dep_next = 0, dep_slot = n3;
        if (tid == 0 && nkind == 2) dep_next = ld_relaxed_gpu(zdone + pb);
        if (kind == 1 && tid == 0 && cb >= nslot) dep_slot = ld_relaxed_gpu(pdone + (cb - nslot));
        if (!issued) {
            // the band of this plane was incomplete at the prefetch point: publish what is pending, then wait for it
            if (pend_z >= 0) {
                if (tid == 0) {
                    asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
                    publish_z(pend_z);
                }
                pend_z = -1;
            }
            if (tid == 0) {
                spin_until_ge(zdone + cb, ntiles);
                issue_input(2, cb, cz, cur, ntiles);
            }
        }
        if (kind == 1) {
            // ================================================================== z tile: packed range -> rows of the ring
            const int band = cur.band;
            const bool act = cur.act;
            const int4 st = cur.st;
            long long a0, a1;
            range_of(cur, a0, a1);
            mbar_wait(&bar_full, par);
            par ^= 1u;
            const long long gs = (mis + (long long)band * pl.S) + st.x;
            const C *src = stage + (gs - a0);
            const int lim = (int)(a1 - gs);
            auto fetch = [&](int idx) -> C {
                if constexpr (EA == 1) return src[idx];
                else return idx < lim ? src[idx] : __ldcs(pk + gs + idx);
            };
            C x[P1], xs[P1];
#pragma unroll
            for (int jj = 0; jj < P1; ++jj) {
                const int idx = ks_of<F>(t, jj) - st.y;
                x[jj] = (act && (unsigned)idx < (unsigned)st.z) ? fetch(idx) : czero<T>();
            }
            const int idb = M / 2 - st.y;
            const C bv = (act && t == 0 && (unsigned)idb < (unsigned)st.z) ? fetch(idb) : czero<T>();
            // the previous z tile's bulk store (thread 0's) must have read the tile before it is overwritten
            if (tid == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncthreads(); // every thread holds its inputs: the landing zone may be refilled, the tile rewritten
            if (tid == 0) s_issued = nkind ? issue_input(nkind, pb, pz, zc, dep_next) : 1;
#pragma unroll
            for (int jj = 0; jj < P1; ++jj) xs[jj] = x[jj];
            xs[P1 / 2] = cadd(xs[P1 / 2], bv);
            C y[B2][P2];
            sub_inv<F, T>(xs, y, tws, zex, t);
#pragma unroll
            for (int bb = 0; bb < B2; ++bb)
#pragma unroll
                for (int q = 0; q < P2; ++q) tile[Z::lin(2 * ((t + P2 * bb) + P1 * q), sl)] = y[bb][q];
            x[P1 / 2] = csub(x[P1 / 2], bv);
            pre_inv<F, 0, T>(x, g);
            sub_inv<F, T>(x, y, tws, zex, t);
#pragma unroll
            for (int bb = 0; bb < B2; ++bb)
#pragma unroll
                for (int q = 0; q < P2; ++q) tile[Z::lin(2 * ((t + P2 * bb) + P1 * q) + 1, sl)] = y[bb][q];
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncthreads();
            issued = s_issued != 0;
            if (tid == 0) {
                if (pend_z >= 0) { // the previous tile is complete in the ring
                    asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
                    publish_z(pend_z);
                }
                // the slot still holds band - nslot until all of its planes have been read
                if (dep_slot < n3) spin_until_ge(pdone + (band - nslot), n3);
                bulk_store_hint(ring + (long long)(band % nslot) * slot_stride + (long long)(cur.s0 / TS) * Z::TILE, tile,
                                (unsigned)(Z::TILE * sizeof(C)), pol_ring);
                asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            }
            pend_z = band;
            prev_z = true;
        } else {
            // ================================================================== plane: row of the ring -> cuboid
            const int b = cb, z = cz;
            if (prev_z) { // the TMA engine must have read the z tile before the plane buffers are written
                if (tid == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
                __syncthreads();
            }
            mbar_wait(&bar_full, par);
            par ^= 1u;
            if (tid == 0) red_relaxed_gpu(pdone + b); // the row is in shared memory: one reader less of its ring slot
            for (int task = warp; task < ntask_y; task += NW) yinv_body(ycol_of(task));
            yinv_single();
            __syncthreads();
            // nobody reads the staged row any more: the next item's input lands during the x pass
            if (tid == 0) {
                s_issued = nkind ? issue_input(nkind, pb, pz, zc, dep_next) : 1;
                if (pend_z >= 0) { // the z tile before this plane has left long ago: complete in the ring
                    asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
                    publish_z(pend_z);
                }
            }
            pend_z = -1;
#pragma unroll
            for (int u = 0; u < XT; ++u) {
                const int v = warp + u * NW, y = v * G + f;
                C *pbuf = (y & 1) ? pb1 : pb0;
                C o0[B2][P2], o1[B2][P2];
                xinv_body(pbuf, y >> 1, o0, o1);
                C *row = cub_out + (((long long)b * n3 + z) * N + y) * N;
                if (hints) {
#pragma unroll
                    for (int bb = 0; bb < B2; ++bb)
#pragma unroll
                        for (int q = 0; q < P2; ++q) st_pair_hint(row + 2 * ((t + P2 * bb) + P1 * q), o0[bb][q], o1[bb][q], pol_stream);
                } else {
#pragma unroll
                    for (int bb = 0; bb < B2; ++bb)
#pragma unroll
                        for (int q = 0; q < P2; ++q) st_pair(row + 2 * ((t + P2 * bb) + P1 * q), o0[bb][q], o1[bb][q]);
                }
            }
            __syncthreads();
            issued = s_issued != 0;
            prev_z = false;
        }
        kind = nkind;
    }
    if (tid == 0 && pend_z >= 0) {
        asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
        publish_z(pend_z);
    }
}

// =====================================================================================================================
// forward
// =====================================================================================================================
template <typename T, class F, int NW>
__global__ void __launch_bounds__(NW * 32, 1)
fused_fwd_k(const __grid_constant__ DevPlan pl, const __grid_constant__ ColTab ct, const cx<T> *__restrict__ cub_in,
            cx<T> *__restrict__ ring, cx<T> *__restrict__ packed, long long slot_stride, int nb, int nslot, int lead,
            int nz, int hints, int *__restrict__ pdone, int *__restrict__ zdone)
{
    using C = cx<T>;
    using FU = Fused<T, F, NW>;
    using PF = typename FU::PF;
    using Z = typename FU::Z;
    constexpr int N = F::N, M = F::M, P1 = F::P1, P2 = F::P2, B2 = F::B2, G = F::G, YP = F::YP;
    constexpr int PB = PF::PB, XT = PF::XT, TS = Z::TS;
    constexpr long long EA = FU::ZP::EA;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int f = lane / P2, t = lane % P2;
    C *const pb0 = reinterpret_cast<C *>(smem_raw), *const pb1 = pb0 + PB; // plane item: [2 residues][NCOL][YP]
    C *const land = pb0 + NW * F::EXW;                                      // z item: exchange tiles, then the packed results
    C *const tile = pb0 + FU::REGP_FWD;                                     // region L, z item: [N/2][RP] (Z::lin)
    C *const lstage = tile + warp * (G * N);                                // region L, plane item: this warp's next G cuboid lines
    __shared__ __align__(8) unsigned long long bar_tile, bar_line[NW];
    __shared__ int s_issued;
    const ExTile<T, P2> zex{pb0 + warp * F::EXW + f * F::FS};
    const int sl = warp * G + f;
    const C *tw = reinterpret_cast<const C *>(pl.tw1); // N1 == N2 == N3: one table
    C tws[P1];
#pragma unroll
    for (int m = 1; m < P1; ++m) tws[m] = tw[modn<N>(2 * t * m)];
    tws[0] = mk<T>((T)1, (T)0);
    const C g = tw[t];
    const T scale = (T)pl.scale;
    const int nx = pl.nxocc, k1lo = pl.k1lo, n3 = pl.n3;
    const bool l0 = (t == 0);
    const int n_one = nx - pl.n_multi;
    const int ntask_y = ycol_tasks<F>(pl.n_multi);
    const long long mis = (long long)(((unsigned long long)packed / sizeof(C)) & (unsigned long long)(EA - 1));
    C *pk = packed - mis;

    const int ntiles = (pl.nsticks + TS - 1) / TS;
    unsigned line_par = 0, tile_par = 0;
    const unsigned long long pol_ring = l2_policy(hints ? 2 : 0), pol_stream = l2_policy(hints ? 1 : 0);
    // stick s of a plane's row inside a ring slot (tile-major), relative to the row's place in tile 0
    auto ring_off = [](int s) -> long long { return (long long)(s / TS) * Z::TILE + (s % TS); };

    // ---- plane item (see plane_pf_k) ----------------------------------------------------------------------------
    struct YCol { bool act; int col; int4 co; };
    auto ycol = [&](int task) -> YCol {
        YCol c;
        const int ci = ycol_index<F>(task, f);
        c.act = task < ntask_y && ci < pl.n_multi;
        c.col = ct.perm[c.act ? ci : 0];
        c.co = ct.col[c.col];
        return c;
    };
    const YCol yc0 = ycol(warp), yc1 = ycol(warp + NW);
    auto ycol_of = [&](int task) -> YCol { return task == warp ? yc0 : task == warp + NW ? yc1 : ycol(task); };
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
    auto xfwd_body = [&](C (&o0)[B2][P2], C (&o1)[B2][P2], C *pbuf, int yl) {
        C g0[P1], g1[P1];
        sub_fwd<F, T>(o0, g0, tws, ExSkew<T, P2, YP>{pbuf + yl, true}, t);
        sub_fwd<F, T>(o1, g1, tws, ExSkew<T, P2, YP>{pbuf + yl, true}, t);
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
    auto yfwd_body = [&](const YCol &c, C *dst) {
        C *pc0 = pb0 + c.col * YP, *pc1 = pb1 + c.col * YP;
        C y[B2][P2], x0[P1], x1[P1];
#pragma unroll
        for (int bb = 0; bb < B2; ++bb)
#pragma unroll
            for (int q = 0; q < P2; ++q) y[bb][q] = pc0[(t + P2 * bb) + P1 * q];
        sub_fwd<F, T>(y, x0, tws, ExSkew<T, P2, 1>{pc0, c.act}, t);
#pragma unroll
        for (int bb = 0; bb < B2; ++bb)
#pragma unroll
            for (int q = 0; q < P2; ++q) y[bb][q] = pc1[(t + P2 * bb) + P1 * q];
        sub_fwd<F, T>(y, x1, tws, ExSkew<T, P2, 1>{pc1, c.act}, t);
        post_fwd<F, 0, T>(x1, g);
        if (c.act) {
            const int idb = M / 2 - c.co.z;
            if (l0 && (unsigned)idb < (unsigned)c.co.y) st_hint(dst + ring_off(c.co.x + idb), csub(x0[P1 / 2], x1[P1 / 2]), pol_ring);
#pragma unroll
            for (int j = 0; j < P1; ++j) {
                const int idx = ks_of<F>(t, j) - c.co.z;
                if ((unsigned)idx < (unsigned)c.co.y) st_hint(dst + ring_off(c.co.x + idx), cadd(x0[j], x1[j]), pol_ring);
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
            if (lane == 0) st_hint(dst + ring_off(co.x), acc, pol_ring);
        }
    };

    // ---- z item (see zpass_pers_fwd_k): descriptor of a tile, loaded one item ahead and not touched before it is needed
    struct ZD { int4 st; int x0, x1, band, s0; bool act; };
    auto describe = [&](int band, int j) -> ZD {
        ZD d;
        d.band = band, d.s0 = j * TS;
        const int s = d.s0 + sl, s1 = d.s0 + TS;
        d.act = s < pl.nsticks;
        d.st = pl.stick[d.act ? s : d.s0];
        d.x0 = pl.stick[d.s0].x;
        d.x1 = s1 < pl.nsticks ? pl.stick[s1].x : (int)pl.S;
        return d;
    };
    // thread 0: the rows of a tile exist once every plane of its band has been written (dep = the counter's value, read
    // earlier); announce their bytes, or return 0 if that is not so yet
    auto expect_tile = [&](const ZD &zd, int dep) -> int {
        if (dep < n3) return 0;
        mbar_expect_tx(&bar_tile, (unsigned)(Z::TILE * sizeof(C)));
        return 1;
    };
    // thread 0 (after expect_tile and a CTA barrier behind the last read of region L): the tile is one contiguous copy
    auto issue_rows = [&](const ZD &zd) {
        if (tid == 0)
            bulk_load_hint(tile, ring + (long long)(zd.band % nslot) * slot_stride + (long long)(zd.s0 / TS) * Z::TILE,
                           (unsigned)(Z::TILE * sizeof(C)), &bar_tile, pol_ring);
    };
    auto line_issue = [&](int b, int z, int v) {
        if (lane == 0) {
            mbar_expect_tx(&bar_line[warp], (unsigned)(G * N * sizeof(C)));
            bulk_load_hint(lstage, cub_in + (((long long)b * n3 + z) * N + (long long)v * G) * N, (unsigned)(G * N * sizeof(C)),
                           &bar_line[warp], pol_stream);
        }
    };

    // this CTA's next tile (band zb, tile zj) and next plane (band pb, plane pz); both lists advance by GD items
    // nz > 0 (spatial split): the first nz CTAs take the z tiles only, the others the planes only
    const int GD = (int)gridDim.x, bid = (int)blockIdx.x;
    const bool zrole = nz > 0 && bid < nz, prole = nz > 0 && bid >= nz;
    const int zs = nz > 0 ? nz : GD, pi = prole ? bid - nz : bid, ps = nz > 0 ? GD - nz : GD;
    int zb = prole ? nb : bid / ntiles, zj = bid % ntiles, pb = zrole ? nb : pi / n3, pz = pi % n3;
    const int dzb = zs / ntiles, dzj = zs % ntiles, dpb = ps / n3, dpz = ps % n3;
    auto peek = [&]() -> int { // 0 none, 1 z tile, 2 plane
        const bool hz = zb < nb, hp = pb < nb;
        if (!hz) return hp ? 2 : 0;
        if (!hp) return 1;
        return zb + lead < pb ? 1 : 2;
    };
    int kind = peek();
    // zc always describes this CTA's next z tile (reloaded when that tile's item starts: nothing waits for the table loads)
    ZD zc = describe(zb < nb ? zb : 0, zb < nb ? zj : 0);
    ZD cur = zc;
    if (tid == 0) {
        mbar_init(&bar_tile, 1);
        for (int w = 0; w < NW; ++w) mbar_init(&bar_line[w], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        s_issued = 0;
    }
    __syncthreads();
    if (kind == 2) line_issue(pb, pz, warp);
    bool prev_z = false; // the previous item was a z tile: its packed bulk store may still be reading region P
    bool issued = false; // the rows of the current item (a z tile) have been requested
    int pend_p = -1;     // band of the last plane whose row has not been published yet (all its stores are behind a CTA barrier)
#pragma unroll 1
    while (kind) {
        const int cb = kind == 1 ? zb : pb, cz = pz;
        if (kind == 1) {
            cur = zc;
            zj += dzj; zb += dzb; if (zj >= ntiles) { zj -= ntiles; ++zb; }
            zc = describe(zb < nb ? zb : 0, zb < nb ? zj : 0);
        } else { pz += dpz; pb += dpb; if (pz >= n3) { pz -= n3; ++pb; } }
        const int nkind = peek();
        // counters this item will look at, read now so that their latency is hidden: the next tile's band (thread 0) and,
        // for a plane, the previous user of its ring slot (lane 0 of every warp)
        int dep_next = 0, dep_slot = ntiles;
        if (tid == 0 && nkind == 1) dep_next = ld_relaxed_gpu(pdone + zb);
        if (kind == 2 && lane == 0 && cb >= nslot) dep_slot = ld_relaxed_gpu(zdone + (cb - nslot));
        if (kind == 2) {
            // ================================================================== plane: cuboid -> row of the ring
            const int b = cb, z = cz;
            if (prev_z) {
                if (tid == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
                __syncthreads();
            }
#pragma unroll
            for (int u = 0; u < XT; ++u) {
                const int v = warp + u * NW, y = v * G + f;
                C o0[B2][P2], o1[B2][P2];
                line_read(o0, o1);
                // the next x task's lines land while this one is transformed
                if (u + 1 < XT) line_issue(b, z, v + NW);
                else if (nkind == 2) line_issue(pb, pz, warp);
                xfwd_body(o0, o1, (y & 1) ? pb1 : pb0, y >> 1);
            }
            if (tid == 0 && nkind == 1) s_issued = expect_tile(zc, dep_next);
            __syncthreads();
            // every warp has read its last lines: the next item's tile may land in region L during the y pass
            issued = nkind == 1 && s_issued != 0;
            if (issued) issue_rows(zc);
            if (tid == 0 && pend_p >= 0) red_release_gpu(pdone + pend_p); // the previous plane's row (stores long drained)
            // the slot still holds band - nslot until all of its tiles have been read
            if (dep_slot < ntiles) spin_until_ge(zdone + (b - nslot), ntiles);
            __syncwarp();
            C *dst = ring + (long long)(b % nslot) * slot_stride + Z::lin(z, 0);
            for (int task = warp; task < ntask_y; task += NW) yfwd_body(ycol_of(task), dst);
            yfwd_single(dst);
            asm volatile("fence.proxy.async.global;" ::: "memory"); // the rows are read by TMA bulk copies of other CTAs
            __syncthreads();
            pend_p = b;
            prev_z = false;
        } else {
            // ================================================================== z tile: rows of the ring -> packed range
            const int band = cur.band;
            const bool act = cur.act;
            const int4 st = cur.st;
            const long long g0 = (mis + (long long)band * pl.S) + cur.x0, g1 = (mis + (long long)band * pl.S) + cur.x1;
            const long long al = g0 & ~(EA - 1), b0 = (g0 + EA - 1) & ~(EA - 1), b1 = g1 & ~(EA - 1);
            if (!issued) { // the band was incomplete at the prefetch point: publish what is pending, then wait for it
                if (tid == 0) {
                    if (pend_p >= 0) red_release_gpu(pdone + pend_p);
                    spin_until_ge(pdone + band, n3);
                    expect_tile(cur, n3);
                }
                pend_p = -1;
                __syncthreads();
                issue_rows(cur);
            }
            mbar_wait(&bar_tile, tile_par);
            tile_par ^= 1u;
            C y[B2][P2], y1[B2][P2], h0[P1], h1[P1];
#pragma unroll
            for (int bb = 0; bb < B2; ++bb)
#pragma unroll
                for (int q = 0; q < P2; ++q) {
                    y[bb][q] = tile[Z::lin(2 * ((t + P2 * bb) + P1 * q), sl)];
                    y1[bb][q] = tile[Z::lin(2 * ((t + P2 * bb) + P1 * q) + 1, sl)];
                }
            if (tid == 0) {
                // the previous tile's packed store must have read the landing zone before it is rewritten
                asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
                red_relaxed_gpu(zdone + band); // the rows are in shared memory: one reader less of the ring slot
                if (pend_p >= 0) red_release_gpu(pdone + pend_p);
                if (nkind == 1) s_issued = expect_tile(zc, dep_next);
            }
            pend_p = -1;
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncthreads(); // every thread holds its tile values: region L may be refilled
            issued = nkind == 1 && s_issued != 0;
            if (issued) issue_rows(zc);
            else if (nkind == 2) line_issue(pb, pz, warp);
            sub_fwd<F, T>(y, h0, tws, zex, t);
            sub_fwd<F, T>(y1, h1, tws, zex, t);
            post_fwd<F, 0, T>(h1, g);
            if (act) {
                const long long gs = (mis + (long long)band * pl.S) + st.x;
                C *dst = land + (gs - al);
                const int lo = (int)(b0 - gs), hi = (int)(b1 - gs); // stick elements [lo, hi) belong to the bulk store
                auto put = [&](int idx, C v) {
                    v = mk<T>(v.x * scale, v.y * scale);
                    if constexpr (EA == 1) dst[idx] = v;
                    else if (idx >= lo && idx < hi) dst[idx] = v;
                    else pk[gs + idx] = v;
                };
                const int idb = M / 2 - st.y;
                if (t == 0 && (unsigned)idb < (unsigned)st.z) put(idb, csub(h0[P1 / 2], h1[P1 / 2]));
#pragma unroll
                for (int jj = 0; jj < P1; ++jj) {
                    const int idx = ks_of<F>(t, jj) - st.y;
                    if ((unsigned)idx < (unsigned)st.z) put(idx, cadd(h0[jj], h1[jj]));
                }
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncthreads();
            if (tid == 0 && b1 > b0) {
                bulk_store_hint(pk + b0, land + (b0 - al), (unsigned)((b1 - b0) * (long long)sizeof(C)), pol_stream);
                asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            }
            prev_z = true;
        }
        kind = nkind;
    }
    if (tid == 0) {
        if (pend_p >= 0) red_release_gpu(pdone + pend_p);
        asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    }
}

} // namespace fftb
