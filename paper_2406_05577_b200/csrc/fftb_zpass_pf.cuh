// fftb_zpass_pf.cuh -- persistent z passes of the fast path (sm_100a).
//
// Inverse: unpack I1 + pruned z-DFT I2 + layout change I3 of SURVEY.md 8(a) (PAPER.md:96 Fig. 3, :112); forward: F5 +
// F6.  Work item = a tile of TS consecutive sticks of one band, one group of P2 lanes per stick (sub_inv / sub_fwd of
// fftb_plane_fast.cuh); the transposition between "one stick, all z" and the plane-major intermediate A[z][stick]
// goes through a shared-memory tile.  Global memory is touched by the TMA engine only:
//   * the packed values of the TS consecutive sticks of a tile are ONE contiguous range of the band (CSR offsets,
//     PAPER.md:183-185); the inverse kernel requests it into a landing zone one tile ahead (cp.async.bulk +
//     mbarrier), so no warp waits for a global load with a scoreboard slot; the forward kernel collects its results
//     there and stores the range with one bulk store;
//   * the rows of the tile leave / arrive as bulk copies (one run of TS elements per z row).
// complex64: a packed range may begin and end on an odd 8-byte element while bulk copies move 16-byte units; loads
// are widened (the neighbours' values are ignored), stores cover the aligned interior and the odd edge elements are
// stored by the lanes that own them.
// A CTA loops over the tiles w = blockIdx.x, blockIdx.x + gridDim.x, ... of the whole batch (w = band * ntiles + j).
#pragma once
#include "fftb_plane_pf.cuh"
#include "fftb_plane_r4.cuh"
#include <cuda.h>

namespace fftb {

template <typename T, class F, int NW> struct ZPers {
    using Z = ZFast<T, F, NW>;
    static constexpr int EA = 16 / (int)sizeof(cx<T>);      // elements per 16 bytes, the granularity of a bulk copy
    static constexpr int LZ = Z::TS * (F::M + 1) + 2 * (EA - 1); // landing zone: TS sticks of at most M + 1 values (+ alignment slack)
    // The tile as the TMA engine's 128-byte swizzle lays it out: per group of SG sticks, N rows (z) of 128 bytes, the 16-byte
    // piece q of row z at piece q ^ (z mod 8).  A tile then leaves / arrives as ONE tensor copy per stick group instead of one
    // bulk copy per z row (the TMA unit takes a copy about every 19 cycles; measured on the 256 pattern, where twice the
    // copies cost 29% and this layout gained 16%), and the transforms' column accesses -- rows two apart, one stick -- stay at
    // most 2-way bank conflicts without padding.  The tile must be 1024-byte aligned.
    static constexpr int SG = 128 / (int)sizeof(cx<T>);      // sticks per 128-byte row: 8 (complex128), 16 (complex64)
    static constexpr int NSG = Z::TS / SG;                   // stick groups (tensor copies) per tile
    static_assert(Z::TS % SG == 0, "tile rows must be whole 128-byte pieces");
    static constexpr int GROUP = F::N * SG;                  // elements of one stick group's part of the tile
    static constexpr int TILE_SW = NSG * GROUP;
    // Row order inside a stick group: the transforms touch the rows z = 2 (t + P2 b + P1 q) + e of one stick with the lanes t
    // of a group side by side, so the tensor the launcher describes splits z into (z / 2) mod 8 | z / 16 | z mod 2 and the
    // box puts (z / 2) mod 8 FASTEST: the 8 (or 4) lanes then hit rows whose low three bits -- what the swizzle XORs into the
    // piece index -- all differ: conflict-free column accesses.
    static_assert(F::N % 16 == 0, "z axis must be a multiple of 16");
    __device__ static __forceinline__ int row(int z) { return ((z & 1) * (F::N / 16) + (z >> 4)) * 8 + ((z >> 1) & 7); }
    __device__ static __forceinline__ int sw(int z, int sl)  // element index of (row z, stick sl of the tile)
    {
        constexpr int PE = 16 / (int)sizeof(cx<T>);          // elements per 16-byte piece
        const int g = sl / SG, s = sl % SG, r = row(z);
        return g * GROUP + r * SG + ((((s / PE) ^ (r & 7)) * PE) | (s % PE));
    }
    static constexpr size_t smem_bytes = sizeof(cx<T>) * ((size_t)TILE_SW + (size_t)NW * F::EXW + (size_t)LZ) + 1024; // + alignment slack
    static constexpr int CTAS_PER_SM = F::P1 > 16 ? 2 : 3;
};

// tile <-> all N3 rows of the sticks x0 / 2 .. of band `band` in A: coordinates of the tensor the launcher builds over the
// intermediate (reals of a row of A | (z / 2) mod 8 | z / 16 | z mod 2 | band), box = {128 bytes, 8, N3 / 16, 2, 1}, 128-byte swizzle
__device__ __forceinline__ void ztile_store(const void *tmap, int x0, int band, const void *ssrc)
{
    asm volatile("cp.async.bulk.tensor.5d.global.shared::cta.tile.bulk_group [%0, {%1, %2, %3, %4, %5}], [%6];" ::"l"(tmap), "r"(x0), "r"(0), "r"(0), "r"(0),
                 "r"(band), "r"((unsigned)__cvta_generic_to_shared(ssrc))
                 : "memory");
}
__device__ __forceinline__ void ztile_load(void *sdst, const void *tmap, int x0, int band, unsigned long long *bar)
{
    asm volatile("cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5, %6}], [%7];" ::"r"(
                     (unsigned)__cvta_generic_to_shared(sdst)),
                 "l"(tmap), "r"(x0), "r"(0), "r"(0), "r"(0), "r"(band), "r"((unsigned)__cvta_generic_to_shared(bar))
                 : "memory");
}

// Batch-fastest packed arrays (BF; Fig. 8 "b x y z": the band index is the fastest one, element
// [point][band] with `pk_pitch` bands per point): the packed range of a tile is no contiguous run of memory any more but
// one element out of every row of pk_pitch.  The kernels stay as they are except for the two places that touch the packed
// array: the landing zone is filled by per-element asynchronous copies (cp.async, completion counted on the same
// mbarrier) and emptied by per-element stores, and the tiles are walked band-fastest (w = tile * bands + band), so that
// the CTAs that run side by side read and write neighbouring elements of the same rows while those are in L2.  The
// transposition [point][band] <-> [band][point] is thereby folded into the z pass; no separate copy of the packed
// arrays is needed (fftb_packed_transpose remains for callers that want one).
__device__ __forceinline__ void cp_async_elem(double2 *sdst, const double2 *gsrc)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(smem_u32(sdst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_elem(float2 *sdst, const float2 *gsrc)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(sdst)), "l"(gsrc) : "memory");
}
// the mbarrier gets this thread's arrival once all of its earlier cp.async copies have landed
__device__ __forceinline__ void cp_async_arrive(unsigned long long *bar)
{
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

template <typename T, class F, int NW, bool BF>
__global__ void __launch_bounds__(NW * 32, ZPers<T, F, NW>::CTAS_PER_SM)
zpass_pers_inv_k(const __grid_constant__ DevPlan pl, const cx<T> *__restrict__ packed, const __grid_constant__ CUtensorMap amap,
                 int ntiles, int total, long long pk_pitch)
{
    using C = cx<T>;
    using Z = ZFast<T, F, NW>;
    using ZP = ZPers<T, F, NW>;
    constexpr int N = F::N, M = F::M, P1 = F::P1, P2 = F::P2, B2 = F::B2, G = F::G, TS = Z::TS, NT = NW * 32;
    constexpr long long EA = BF ? 1 : ZPers<T, F, NW>::EA;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // `packed` may be only 8-byte aligned (complex64 band chunks of the library's own calls): indices below count
    // elements from the 16-byte boundary pk at or below it
    const long long mis = BF ? 0 : (long long)(((unsigned long long)packed / sizeof(C)) & (unsigned long long)(EA - 1));
    const C *pk = packed - mis;
    unsigned char *t_raw = smem_raw + ((1024u - ((unsigned)__cvta_generic_to_shared(smem_raw) & 1023u)) & 1023u);
    C *tile = reinterpret_cast<C *>(t_raw);               // [stick group][N][SG], 128-byte swizzle (ZPers::sw)
    C *land = tile + ZP::TILE_SW + NW * F::EXW;           // packed values of the tile's sticks
    __shared__ __align__(8) unsigned long long bar;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int f = lane / P2, t = lane % P2;
    const ExTile<T, P2> ex{tile + ZP::TILE_SW + warp * F::EXW + f * F::FS};
    const int sl = warp * G + f;
    const C *tw = reinterpret_cast<const C *>(pl.tw3);
    C tws[P1];
#pragma unroll
    for (int m = 1; m < P1; ++m) tws[m] = tw[modn<N>(2 * t * m)];
    tws[0] = mk<T>((T)1, (T)0);
    const C g = tw[t];
    const int nbands = total / ntiles;

    // Descriptor of tile w, loaded one iteration before it is used (the stick table is in global memory): this
    // lane's stick and the packed range of the tile in elements of the whole batch, widened to 16-byte boundaries
    // [a0, a1) (complex64: a range may begin and end on an odd element; the neighbours' values that come along are
    // not used).  The batch ends at nall: an odd last element is not covered (a1 < end of the range) and is read
    // straight from global.  BF: the range counts points of one band, [a0, a1) = the tile's points exactly.
    const long long nall = mis + (long long)nbands * pl.S;
    struct Tile { int4 st; long long a0, a1; int band, s0; bool act; };
    auto describe = [&](int w) -> Tile {
        Tile d;
        if constexpr (BF) d.band = w % nbands, d.s0 = (w / nbands) * TS;
        else d.band = w / ntiles, d.s0 = (w % ntiles) * TS;
        const int s = d.s0 + sl, s1 = d.s0 + TS;
        d.act = s < pl.nsticks;
        d.st = pl.stick[d.act ? s : d.s0]; // {off, k3lo, len, .}
        const long long base = BF ? 0 : mis + (long long)d.band * pl.S;
        const long long g0 = base + pl.stick[d.s0].x;
        const long long g1 = base + (s1 < pl.nsticks ? (long long)pl.stick[s1].x : pl.S);
        d.a0 = g0 & ~(EA - 1);
        d.a1 = (g1 + EA - 1) & ~(EA - 1);
        if (!BF && d.a1 > nall) d.a1 = nall & ~(EA - 1);
        return d;
    };
    // ask for the packed range of a tile: thread 0 with one bulk copy, or (BF) every thread with its share of elements
    auto issue = [&](const Tile &d) {
        if constexpr (BF) {
            const C *src = packed + d.a0 * pk_pitch + d.band;
            const int n = (int)(d.a1 - d.a0);
            for (int i = tid; i < n; i += NT) cp_async_elem(land + i, src + (long long)i * pk_pitch);
            cp_async_arrive(&bar);
        } else if (tid == 0) {
            const unsigned bytes = (unsigned)((d.a1 - d.a0) * (long long)sizeof(C));
            mbar_expect_tx(&bar, bytes);
            if (bytes) bulk_load(land, pk + d.a0, bytes, &bar); // 0: a single odd last element of the batch, read directly
        }
    };
    if (tid == 0) {
        mbar_init(&bar, BF ? NT : 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    int w = blockIdx.x;
    Tile cur = describe(w < total ? w : 0), nxt = cur;
    if (w < total) issue(cur);
    unsigned par = 0;
#pragma unroll 1
    for (; w < total; w += gridDim.x) {
        const bool more = w + (int)gridDim.x < total;
        if (more) nxt = describe(w + (int)gridDim.x);
        const int band = cur.band, s0 = cur.s0;
        const bool act = cur.act;
        const int4 st = cur.st;
        const long long a0 = cur.a0, a1 = cur.a1;
        mbar_wait(&bar, par);
        par ^= 1u;
        const long long gs = (BF ? 0 : mis + (long long)band * pl.S) + st.x; // the stick's first element
        const C *src = land + (gs - a0);
        const int lim = (int)(a1 - gs);                      // elements of the stick from here on are not in the landing zone
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
        // the previous tile's tensor copies (thread 0's) must have read the tile before it is overwritten
        if (tid == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads(); // every thread holds its inputs: the landing zone may be refilled, the tile rewritten
        if (more) issue(nxt);
#pragma unroll
        for (int jj = 0; jj < P1; ++jj) xs[jj] = x[jj];
        xs[P1 / 2] = cadd(xs[P1 / 2], bv);
        C y[B2][P2];
        sub_inv<F, T>(xs, y, tws, ex, t);
#pragma unroll
        for (int bb = 0; bb < B2; ++bb)
#pragma unroll
            for (int q = 0; q < P2; ++q) tile[ZP::sw(2 * ((t + P2 * bb) + P1 * q), sl)] = y[bb][q];
        x[P1 / 2] = csub(x[P1 / 2], bv);
        pre_inv<F, 0, T>(x, g);
        sub_inv<F, T>(x, y, tws, ex, t);
#pragma unroll
        for (int bb = 0; bb < B2; ++bb)
#pragma unroll
            for (int q = 0; q < P2; ++q) tile[ZP::sw(2 * ((t + P2 * bb) + P1 * q) + 1, sl)] = y[bb][q];
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();
        // one tensor copy per group of SG sticks (groups beyond the row pitch do not exist)
        if (tid == 0) {
#pragma unroll
            for (int gq = 0; gq < ZP::NSG; ++gq)
                if (s0 + gq * ZP::SG < pl.pitch) ztile_store(&amap, (s0 + gq * ZP::SG) * (int)(sizeof(C) / sizeof(T)), band, tile + gq * ZP::GROUP);
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
        cur = nxt;
    }
    if (tid == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

// Forward (F5 z-DFT keeping the stick's k3, scale, F6 pack): the N rows A[z][s0 .. s0 + TS) of the next tile are
// requested as bulk loads as soon as every thread holds its tile values; the results of a tile are collected in the
// landing zone in packed order and leave as ONE bulk store (the packed range of TS consecutive sticks is contiguous),
// or (BF) as per-element stores into the batch-fastest array.  Only for one plane of A (ry == 1).
template <typename T, class F, int NW, bool BF>
__global__ void __launch_bounds__(NW * 32, ZPers<T, F, NW>::CTAS_PER_SM)
zpass_pers_fwd_k(const __grid_constant__ DevPlan pl, const __grid_constant__ CUtensorMap amap, cx<T> *__restrict__ packed,
                 int ntiles, int total, long long pk_pitch)
{
    using C = cx<T>;
    using Z = ZFast<T, F, NW>;
    using ZP = ZPers<T, F, NW>;
    constexpr int N = F::N, M = F::M, P1 = F::P1, P2 = F::P2, B2 = F::B2, G = F::G, TS = Z::TS, NT = NW * 32;
    constexpr long long EA = BF ? 1 : ZPers<T, F, NW>::EA;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // `packed` may be only 8-byte aligned (complex64 band chunks of the library's own calls): indices below count
    // elements from the 16-byte boundary pk at or below it
    const long long mis = BF ? 0 : (long long)(((unsigned long long)packed / sizeof(C)) & (unsigned long long)(EA - 1));
    C *pk = packed - mis;
    unsigned char *t_raw = smem_raw + ((1024u - ((unsigned)__cvta_generic_to_shared(smem_raw) & 1023u)) & 1023u);
    C *tile = reinterpret_cast<C *>(t_raw);               // [stick group][N][SG], 128-byte swizzle (ZPers::sw)
    C *land = tile + ZP::TILE_SW + NW * F::EXW;           // results of the tile's sticks in packed order
    __shared__ __align__(8) unsigned long long bar;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int f = lane / P2, t = lane % P2;
    const ExTile<T, P2> ex{tile + ZP::TILE_SW + warp * F::EXW + f * F::FS};
    const int sl = warp * G + f;
    const C *tw = reinterpret_cast<const C *>(pl.tw3);
    C tws[P1];
#pragma unroll
    for (int m = 1; m < P1; ++m) tws[m] = tw[modn<N>(2 * t * m)];
    tws[0] = mk<T>((T)1, (T)0);
    const C g = tw[t];
    const T scale = (T)pl.scale;
    const int nbands = total / ntiles;
    auto band_of = [&](int w) { return BF ? w % nbands : w / ntiles; };
    auto s0_of = [&](int w) { return (BF ? w / nbands : w % ntiles) * TS; };

    // thread 0 announces the bytes of tile w and asks for it: one tensor copy per group of SG sticks (groups beyond the row
    // pitch do not exist; their part of the tile is never looked at by an active stick)
    auto issue_rows = [&](int w) {
        if (tid == 0) {
            const int band = band_of(w), s0 = s0_of(w);
            int ng = 0;
#pragma unroll
            for (int gq = 0; gq < ZP::NSG; ++gq) ng += (s0 + gq * ZP::SG < pl.pitch) ? 1 : 0;
            mbar_expect_tx(&bar, (unsigned)(ng * ZP::GROUP * (int)sizeof(C)));
#pragma unroll
            for (int gq = 0; gq < ZP::NSG; ++gq)
                if (s0 + gq * ZP::SG < pl.pitch) ztile_load(tile + gq * ZP::GROUP, &amap, (s0 + gq * ZP::SG) * (int)(sizeof(C) / sizeof(T)), band, &bar);
        }
    };
    if (tid == 0) {
        mbar_init(&bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    int w = blockIdx.x;
    if (w < total) issue_rows(w);
    unsigned par = 0;
#pragma unroll 1
    for (; w < total; w += gridDim.x) {
        const bool more = w + (int)gridDim.x < total;
        const int band = band_of(w), s0 = s0_of(w), s = s0 + sl;
        const bool act = s < pl.nsticks;
        const int4 st = pl.stick[act ? s : s0];
        // the tile's packed range [g0, g1) in elements of the whole batch (used after the transforms: loading the table
        // one tile ahead was measured 3% slower); its 16-byte aligned interior [b0, b1) leaves as one bulk store from the
        // landing zone (origin al), an odd first / last element (complex64) by a plain store.  BF: points of one band.
        const long long base = BF ? 0 : mis + (long long)band * pl.S;
        const long long g0 = base + pl.stick[s0].x;
        const long long g1 = base + (s0 + TS < pl.nsticks ? (long long)pl.stick[s0 + TS].x : pl.S);
        const long long al = g0 & ~(EA - 1), b0 = (g0 + EA - 1) & ~(EA - 1), b1 = g1 & ~(EA - 1);
        mbar_wait(&bar, par);
        par ^= 1u;
        C y[B2][P2], y1[B2][P2], h0[P1], h1[P1];
#pragma unroll
        for (int bb = 0; bb < B2; ++bb)
#pragma unroll
            for (int q = 0; q < P2; ++q) {
                y[bb][q] = tile[ZP::sw(2 * ((t + P2 * bb) + P1 * q), sl)];
                y1[bb][q] = tile[ZP::sw(2 * ((t + P2 * bb) + P1 * q) + 1, sl)];
            }
        // the previous tile's packed store must have read the landing zone before it is rewritten
        if (tid == 0) {
            if constexpr (!BF) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads(); // every thread holds its tile values: the next tile's rows may land
        if (more) issue_rows(w + (int)gridDim.x);
        sub_fwd<F, T>(y, h0, tws, ex, t);
        sub_fwd<F, T>(y1, h1, tws, ex, t);
        post_fwd<F, 0, T>(h1, g);
        if (act) {
            const long long gs = base + st.x;
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
        if constexpr (BF) {
            // the tile's points, one element out of every row of the batch-fastest array (the next write to the landing
            // zone comes after the next CTA barrier, which this thread only reaches once its loop is done)
            C *out = packed + g0 * pk_pitch + band;
            const int n = (int)(g1 - g0);
            for (int i = tid; i < n; i += NT) out[(long long)i * pk_pitch] = land[i];
        } else if (tid == 0 && b1 > b0) {
            bulk_store(pk + b0, land + (b0 - al), (unsigned)((b1 - b0) * (long long)sizeof(C)));
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
    }
    if (tid == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}

// ---------------------------------------------------------------------------------------------
// 256 pattern (four-way split z = 4 n' + e, fftb_plane_r4.cuh): the same persistent schedule, but a tile of all 256
// rows (66 KB) next to the landing zone (16 x 129 values) would leave one CTA per SM, so the shared-memory tile
// holds HALF of the rows: the residues e = 0, 1 are transformed, written and sent; the residues e = 2, 3 are
// transformed while the TMA engine reads the tile and take its place.  Row (n', e & 1) of a half sits at
// n' RP + (e & 1) TS (ZFast::lin with z = 2 n' + (e & 1)).
// ---------------------------------------------------------------------------------------------
template <typename T, int NW> struct ZPersR4 {
    using F = FastCfg<T, 128, 8, 8>;
    using Z = ZFast<T, F, NW>;                               // tile of 128 rows = half of the 256
    static constexpr int N = 256, M = 64, TS = Z::TS;
    static constexpr int EA = 16 / (int)sizeof(cx<T>);
    static constexpr int LZ = TS * (2 * M + 1) + 2 * (EA - 1);
    // The half tile as the TMA engine's 128-byte swizzle lays it out: 2 M rows (n', e & 1) of 128 bytes per group of SG
    // sticks, the 16-byte piece q of row r at piece q ^ (r mod 8).  A half tile then leaves / arrives as ONE tensor copy per
    // stick group instead of one bulk copy per row (the TMA unit takes a copy about every 19 cycles: 256 row copies per tile
    // were most of the tile's time), and the transforms' column accesses -- rows two apart, one stick -- are 2-way instead of
    // 8-way bank conflicts without any padding.  The tile must be 1024-byte aligned.
    static constexpr int SG = 128 / (int)sizeof(cx<T>);      // sticks per 128-byte row: 8 (complex128), 16 (complex64)
    static constexpr int NSG = TS / SG;                      // stick groups (tensor copies) per half tile
    static_assert(TS % SG == 0, "tile rows must be whole 128-byte pieces");
    static constexpr int HALF = 2 * M * SG;                  // elements of one stick group's half tile (16 KB)
    static constexpr int TILE_SW = NSG * HALF;
    // row r = 2 n' + (e & 1) of the half sits at ((e & 1) 8 + n' / 8) 8 + n' mod 8: n' mod 8 fastest, see ZPers::row
    __device__ static __forceinline__ int sw(int rr, int sl) // element index of (row rr of the half, stick sl of the tile)
    {
        constexpr int PE = 16 / (int)sizeof(cx<T>);          // elements per 16-byte piece
        const int g = sl / SG, s = sl % SG, r = ((rr & 1) * 8 + (rr >> 4)) * 8 + ((rr >> 1) & 7);
        return g * HALF + r * SG + ((((s / PE) ^ (r & 7)) * PE) | (s % PE));
    }
    static constexpr size_t smem_bytes = sizeof(cx<T>) * ((size_t)TILE_SW + (size_t)NW * F::EXW + (size_t)LZ) + 1024; // + alignment slack
};

// half tile <-> the rows z = 4 n' + e0, 4 n' + e0 + 1 of the sticks s0 + SG g .. of band `band` in A: coordinates of the tensor
// the launcher builds over the intermediate (reals of SG sticks | n' mod 8 | n' / 8 | z mod 4 | band), box = {128 bytes, 8, 8, 2, 1}
__device__ __forceinline__ void zr4_half_store(const void *tmap, int x0, int e0, int band, const void *ssrc)
{
    asm volatile("cp.async.bulk.tensor.5d.global.shared::cta.tile.bulk_group [%0, {%1, %2, %3, %4, %5}], [%6];" ::"l"(tmap), "r"(x0), "r"(0), "r"(0), "r"(e0),
                 "r"(band), "r"(smem_u32(ssrc))
                 : "memory");
}
__device__ __forceinline__ void zr4_half_load(void *sdst, const void *tmap, int x0, int e0, int band, unsigned long long *bar)
{
    asm volatile("cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5, %6}], [%7];" ::"r"(smem_u32(sdst)),
                 "l"(tmap), "r"(x0), "r"(0), "r"(0), "r"(e0), "r"(band), "r"(smem_u32(bar))
                 : "memory");
}

template <typename T, int NW>
__global__ void __launch_bounds__(NW * 32, 2)
zpass_r4_pers_inv_k(const __grid_constant__ DevPlan pl, const cx<T> *__restrict__ packed, const __grid_constant__ CUtensorMap amap,
                    int ntiles, int total)
{
    using C = cx<T>;
    using ZP = ZPersR4<T, NW>;
    using F = typename ZP::F;
    using Z = typename ZP::Z;
    constexpr int M = ZP::M, P2 = F::P2, G = F::G, TS = ZP::TS, NT = NW * 32;
    constexpr long long EA = ZP::EA;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // `packed` may be only 8-byte aligned (complex64 band chunks of the library's own calls): indices below count
    // elements from the 16-byte boundary pk at or below it
    const long long mis = (long long)(((unsigned long long)packed / sizeof(C)) & (unsigned long long)(EA - 1));
    const C *pk = packed - mis;
    unsigned char *t_raw = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    C *tile = reinterpret_cast<C *>(t_raw);               // half tile: rows (n', e & 1), 128-byte swizzle (ZPersR4::sw)
    C *land = tile + ZP::TILE_SW + NW * F::EXW;           // packed values of the tile's sticks
    __shared__ __align__(8) unsigned long long bar;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int f = lane / P2, t = lane % P2;
    const ExTile<T, P2> ex{tile + ZP::TILE_SW + warp * F::EXW + f * F::FS};
    const int sl = warp * G + f;
    const C *tw = reinterpret_cast<const C *>(pl.tw3);
    C tws[8], wt[4];
#pragma unroll
    for (int m = 1; m < 8; ++m) tws[m] = tw[(4 * t * m) & (ZP::N - 1)];
    tws[0] = mk<T>((T)1, (T)0);
#pragma unroll
    for (int e = 0; e < 4; ++e) wt[e] = tw[e * t];

    const long long nall = mis + (long long)(total / ntiles) * pl.S;
    auto range = [&](int w, long long &a0, long long &a1) { // see zpass_pers_inv_k
        const int band = w / ntiles, s0 = (w % ntiles) * TS, s1 = s0 + TS;
        const long long g0 = (mis + (long long)band * pl.S) + pl.stick[s0].x;
        const long long g1 = (mis + (long long)band * pl.S) + (s1 < pl.nsticks ? (long long)pl.stick[s1].x : pl.S);
        a0 = g0 & ~(EA - 1);
        a1 = (g1 + EA - 1) & ~(EA - 1);
        if (a1 > nall) a1 = nall & ~(EA - 1);
    };
    auto issue = [&](int w) {
        long long a0, a1;
        range(w, a0, a1);
        const unsigned bytes = (unsigned)((a1 - a0) * (long long)sizeof(C));
        mbar_expect_tx(&bar, bytes);
        if (bytes) bulk_load(land, pk + a0, bytes, &bar); // 0: a single odd last element of the batch, read directly
    };
    if (tid == 0) {
        mbar_init(&bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    int w = blockIdx.x;
    if (tid == 0 && w < total) issue(w);
    unsigned par = 0;
#pragma unroll 1
    for (; w < total; w += gridDim.x) {
        const int band = w / ntiles, s0 = (w % ntiles) * TS, s = s0 + sl;
        const bool act = s < pl.nsticks;
        const int4 st = pl.stick[act ? s : s0]; // {off, k3lo, len, .}
        long long a0, a1;
        range(w, a0, a1);
        mbar_wait(&bar, par);
        par ^= 1u;
        const long long gs = (mis + (long long)band * pl.S) + st.x;
        const C *src = land + (gs - a0);
        const int lim = (int)(a1 - gs);
        auto fetch = [&](int idx) -> C {
            if constexpr (EA == 1) return src[idx];
            else return idx < lim ? src[idx] : __ldcs(pk + gs + idx);
        };
        C a[8], bq[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const int ia = (t + 8 * j) - M - st.y, ib = (t + 8 * j) - st.y;
            a[j] = (act && (unsigned)ia < (unsigned)st.z) ? fetch(ia) : czero<T>();
            bq[j] = (act && (unsigned)ib < (unsigned)st.z) ? fetch(ib) : czero<T>();
        }
        const int ic = M - st.y;
        const C cv = (act && t == 0 && (unsigned)ic < (unsigned)st.z) ? fetch(ic) : czero<T>();
        // the previous tile's second half must have left the tile (thread 0 issued the copies)
        if (tid == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads(); // every thread holds its inputs: the landing zone may be refilled, the tile rewritten
        if (tid == 0 && w + (int)gridDim.x < total) issue(w + (int)gridDim.x);
        // rows z = 4 n' + e0 + (r & 1), n' = r >> 1, of the half in the tile: one tensor copy per group of SG sticks
        auto send_half = [&](int e0) {
            if (tid == 0) {
#pragma unroll
                for (int g = 0; g < ZP::NSG; ++g)
                    zr4_half_store(&amap, (s0 + g * ZP::SG) * (int)(sizeof(C) / sizeof(T)), e0, band, tile + g * ZP::HALF);
                asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            }
        };
        C u[8], y[1][8], y2[1][8];
        r4_fold_inv<0, 0, T>(a, bq, cv, u, wt[0]);
        sub_inv<F, T>(u, y, tws, ex, t);
#pragma unroll
        for (int q = 0; q < 8; ++q) tile[ZP::sw(2 * (t + 8 * q), sl)] = y[0][q];
        r4_fold_inv<1, 0, T>(a, bq, cv, u, wt[1]);
        sub_inv<F, T>(u, y, tws, ex, t);
#pragma unroll
        for (int q = 0; q < 8; ++q) tile[ZP::sw(2 * (t + 8 * q) + 1, sl)] = y[0][q];
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();
        send_half(0);
        r4_fold_inv<2, 0, T>(a, bq, cv, u, wt[2]);
        sub_inv<F, T>(u, y, tws, ex, t);
        r4_fold_inv<3, 0, T>(a, bq, cv, u, wt[3]);
        sub_inv<F, T>(u, y2, tws, ex, t);
        if (tid == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        __syncthreads(); // the first half has left
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            tile[ZP::sw(2 * (t + 8 * q), sl)] = y[0][q];
            tile[ZP::sw(2 * (t + 8 * q) + 1, sl)] = y2[0][q];
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();
        send_half(2);
    }
    if (tid == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

// forward z pass of the 256 pattern (one plane of A): the rows of the residues e = 0, 1 and e = 2, 3 arrive in the half
// tile one after the other, each requested as soon as every thread holds the values of the half before it
template <typename T, int NW>
__global__ void __launch_bounds__(NW * 32, 2)
zpass_r4_pers_fwd_k(const __grid_constant__ DevPlan pl, const __grid_constant__ CUtensorMap amap, cx<T> *__restrict__ packed,
                    int ntiles, int total)
{
    using C = cx<T>;
    using ZP = ZPersR4<T, NW>;
    using F = typename ZP::F;
    using Z = typename ZP::Z;
    constexpr int M = ZP::M, P2 = F::P2, G = F::G, TS = ZP::TS, NT = NW * 32;
    constexpr long long EA = ZP::EA;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // `packed` may be only 8-byte aligned (complex64 band chunks of the library's own calls): indices below count
    // elements from the 16-byte boundary pk at or below it
    const long long mis = (long long)(((unsigned long long)packed / sizeof(C)) & (unsigned long long)(EA - 1));
    C *pk = packed - mis;
    unsigned char *t_raw = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    C *tile = reinterpret_cast<C *>(t_raw);               // half tile: rows (n', e & 1), 128-byte swizzle (ZPersR4::sw)
    C *land = tile + ZP::TILE_SW + NW * F::EXW;           // results of the tile's sticks in packed order
    __shared__ __align__(8) unsigned long long bar;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int f = lane / P2, t = lane % P2;
    const ExTile<T, P2> ex{tile + ZP::TILE_SW + warp * F::EXW + f * F::FS};
    const int sl = warp * G + f;
    const C *tw = reinterpret_cast<const C *>(pl.tw3);
    C tws[8], wt[4];
#pragma unroll
    for (int m = 1; m < 8; ++m) tws[m] = tw[(4 * t * m) & (ZP::N - 1)];
    tws[0] = mk<T>((T)1, (T)0);
#pragma unroll
    for (int e = 0; e < 4; ++e) wt[e] = tw[e * t];
    const T scale = (T)pl.scale;

    // thread 0 announces the bytes of a half of tile w and asks for it: one tensor copy per group of SG sticks
    auto issue_half = [&](int w, int e0) {
        if (tid == 0) {
            const int band = w / ntiles, s0 = (w % ntiles) * TS;
            mbar_expect_tx(&bar, (unsigned)(ZP::TILE_SW * sizeof(C)));
#pragma unroll
            for (int g = 0; g < ZP::NSG; ++g)
                zr4_half_load(tile + g * ZP::HALF, &amap, (s0 + g * ZP::SG) * (int)(sizeof(C) / sizeof(T)), e0, band, &bar);
        }
    };
    if (tid == 0) {
        mbar_init(&bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    int w = blockIdx.x;
    if (w < total) issue_half(w, 0);
    unsigned par = 0;
#pragma unroll 1
    for (; w < total; w += gridDim.x) {
        const bool more = w + (int)gridDim.x < total;
        const int band = w / ntiles, s0 = (w % ntiles) * TS, s = s0 + sl;
        const bool act = s < pl.nsticks;
        const int4 st = pl.stick[act ? s : s0];
        const long long g0 = (mis + (long long)band * pl.S) + pl.stick[s0].x;
        const long long g1 = (mis + (long long)band * pl.S) + (s0 + TS < pl.nsticks ? (long long)pl.stick[s0 + TS].x : pl.S);
        const long long al = g0 & ~(EA - 1), b0 = (g0 + EA - 1) & ~(EA - 1), b1 = g1 & ~(EA - 1); // see zpass_pers_fwd_k
        C y[1][8], y2[1][8], gq[8], fa[8], fb[8], fc;
        // ---- residues e = 0, 1
        mbar_wait(&bar, par);
        par ^= 1u;
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            y[0][q] = tile[ZP::sw(2 * (t + 8 * q), sl)];
            y2[0][q] = tile[ZP::sw(2 * (t + 8 * q) + 1, sl)];
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads(); // every thread holds its values: the other half of the rows may land
        issue_half(w, 2);
        sub_fwd<F, T>(y, gq, tws, ex, t);
        r4_fold_fwd<0, 0, T>(gq, fa, fb, fc, wt[0]);
        sub_fwd<F, T>(y2, gq, tws, ex, t);
        r4_fold_fwd<1, 0, T>(gq, fa, fb, fc, wt[1]);
        // ---- residues e = 2, 3
        mbar_wait(&bar, par);
        par ^= 1u;
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            y[0][q] = tile[ZP::sw(2 * (t + 8 * q), sl)];
            y2[0][q] = tile[ZP::sw(2 * (t + 8 * q) + 1, sl)];
        }
        // the previous tile's packed store must have read the landing zone before it is rewritten
        if (tid == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();
        if (more) issue_half(w + (int)gridDim.x, 0);
        sub_fwd<F, T>(y, gq, tws, ex, t);
        r4_fold_fwd<2, 0, T>(gq, fa, fb, fc, wt[2]);
        sub_fwd<F, T>(y2, gq, tws, ex, t);
        r4_fold_fwd<3, 0, T>(gq, fa, fb, fc, wt[3]);
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
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const int ia = (t + 8 * j) - M - st.y, ib = (t + 8 * j) - st.y;
                if ((unsigned)ia < (unsigned)st.z) put(ia, fa[j]);
                if ((unsigned)ib < (unsigned)st.z) put(ib, fb[j]);
            }
            const int ic = M - st.y;
            if (t == 0 && (unsigned)ic < (unsigned)st.z) put(ic, fc);
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();
        if (tid == 0 && b1 > b0) {
            bulk_store(pk + b0, land + (b0 - al), (unsigned)((b1 - b0) * (long long)sizeof(C)));
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
    }
    if (tid == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}

} // namespace fftb
