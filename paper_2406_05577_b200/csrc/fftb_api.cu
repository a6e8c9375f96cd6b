// fftb_api.cu -- host plan builder, kernel dispatch and the C-ABI of include/fftb.h.
//
// The plan builder is the paper's "computational layout descriptor" + "transform creation"
// blocks collapsed for one GPU: it turns the bounding domain (N1,N2,N3), the
// cut-off and the batch size into the offset array (stick map, Fig. 7, 183-185) and
// the per-k1 stick runs, picks one of the predefined kernel patterns or refuses
// (FFTB_EUNSUPPORTED), and sizes the workspace.
#include "../../include/fftb.h"
#include "fftb_kernels.cuh"
#include "fftb_plane_fast.cuh"
#include "fftb_plane_pf.cuh"
#include "fftb_plane_r4.cuh"
#include "fftb_zpass_pf.cuh"
#include "fftb_fused.cuh"
#include "fftb_dense.cuh"
#include "fftb_probe.cuh"
#include "fftb_slab.cuh"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <utility>
#include <vector>

using namespace fftb;

namespace {

// ------------------------------------------------------------------------------------------------
// predefined patterns: axis length -> factorisation
// ------------------------------------------------------------------------------------------------
template <int N, bool DENSE> struct ZX; // z and x axes: the R sub-transforms are done by one thread group
template <> struct ZX<32, false> { using type = Axis<32, 2, 4, 4, true>; };
template <> struct ZX<64, false> { using type = Axis<64, 2, 8, 4, true>; };
template <> struct ZX<96, false> { using type = Axis<96, 2, 6, 8, true>; };
template <> struct ZX<128, false> { using type = Axis<128, 2, 8, 8, true>; };
template <> struct ZX<192, false> { using type = Axis<192, 2, 12, 8, true>; };
template <> struct ZX<256, false> { using type = Axis<256, 2, 16, 8, true>; };
template <> struct ZX<32, true> { using type = Axis<32, 1, 8, 4, false>; };
template <> struct ZX<64, true> { using type = Axis<64, 1, 8, 8, false>; };
template <> struct ZX<128, true> { using type = Axis<128, 1, 16, 8, false>; };
template <> struct ZX<256, true> { using type = Axis<256, 1, 16, 16, false>; };

template <int N, bool DENSE> struct YA; // y axis: the R residues go to R different CTAs
template <> struct YA<32, false> { using type = Axis<32, 2, 4, 4, true>; };
template <> struct YA<64, false> { using type = Axis<64, 2, 8, 4, true>; };
template <> struct YA<96, false> { using type = Axis<96, 2, 6, 8, true>; };
template <> struct YA<128, false> { using type = Axis<128, 2, 8, 8, true>; };
template <> struct YA<192, false> { using type = Axis<192, 4, 6, 8, true>; };
template <> struct YA<256, false> { using type = Axis<256, 4, 8, 8, true>; };
template <> struct YA<32, true> { using type = Axis<32, 1, 8, 4, false>; };
template <> struct YA<64, true> { using type = Axis<64, 1, 8, 8, false>; };
template <> struct YA<128, true> { using type = Axis<128, 2, 8, 8, false>; };
template <> struct YA<256, true> { using type = Axis<256, 8, 8, 4, false>; };

constexpr int cmax(int a, int b) { return a > b ? a : b; }
// largest divisor of m that does not exceed cap
constexpr int div_le(int m, int cap)
{
    int best = 1;
    for (int d = 1; d <= m && d <= cap; ++d)
        if (m % d == 0) best = d;
    return best;
}

template <class AX, class AY> struct PlaneTune {
    static constexpr int PM = cmax(AX::P1, AX::P2);
    static constexpr int LX = div_le(AY::M, 256 / PM);          // lines per x round
    static constexpr int NT = LX * PM;                         // threads per CTA
    static constexpr int LY = cmax(1, NT / cmax(AY::P1, AY::P2)); // columns per y round
};

constexpr int Z_LINES = 32, Z_NT = 256;

// ------------------------------------------------------------------------------------------------
// Launch-side state.  Nothing here depends on the calling thread or on a previous launch: the one piece of
// per-kernel device state (the opt-in limit on dynamic shared memory) is raised ONCE per (kernel, device) to the
// device's maximum under a mutex and never lowered, the occupancy of a (kernel, device, shared memory) triple is
// cached in the same registry, and the SM count of the device a plan was bound on travels in its DevPlan.
// ------------------------------------------------------------------------------------------------
struct KernelState {
    bool attr_set = false;
    std::map<size_t, int> per_sm; // dynamic shared memory -> resident CTAs per SM
};
std::mutex g_reg_mu;
std::map<std::pair<const void *, int>, KernelState> g_reg;

int current_device()
{
    int dev = 0;
    cudaGetDevice(&dev);
    return dev;
}

// makes kernel k launchable with `smem` bytes of dynamic shared memory on the current device; per_sm (optional)
// receives the number of CTAs of `threads` threads that fit one SM
int kernel_ready(const void *k, int threads, size_t smem, int *per_sm)
{
    const int dev = current_device();
    std::lock_guard<std::mutex> lock(g_reg_mu);
    KernelState &ks = g_reg[std::make_pair(k, dev)];
    if (!ks.attr_set) {
        int optin = 0;
        cudaFuncAttributes fa;
        if (cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess) return FFTB_ECUDA;
        if (cudaFuncGetAttributes(&fa, k) != cudaSuccess) return FFTB_ECUDA;
        // static + dynamic shared memory of a block may not exceed the opt-in limit
        const int dyn_max = optin - (int)fa.sharedSizeBytes;
        if (dyn_max < 0 || cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, dyn_max) != cudaSuccess) {
            cudaGetLastError();
            return FFTB_ECUDA;
        }
        ks.attr_set = true;
    }
    if (per_sm) {
        auto it = ks.per_sm.find(smem);
        if (it == ks.per_sm.end()) {
            int occ = 0;
            if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k, threads, smem) != cudaSuccess) return FFTB_ECUDA;
            it = ks.per_sm.emplace(smem, occ).first;
        }
        *per_sm = it->second;
        if (*per_sm < 1) return FFTB_EUNSUPPORTED;
    }
    return 0;
}
template <class K> int kernel_ready(K k, int threads, size_t smem, int *per_sm)
{
    return kernel_ready(reinterpret_cast<const void *>(k), threads, smem, per_sm);
}
int launch_status() { return cudaGetLastError() == cudaSuccess ? 0 : FFTB_ECUDA; }

struct ZLaunch {
    // pk_pitch: 0 = packed [band][point]; > 0 = batch-fastest packed [point][pk_pitch bands] (persistent TMA z kernels only)
    int (*inv)(const DevPlan &, const void *packed, void *A, long long stride, int nb, long long pk_pitch, cudaStream_t);
    int (*fwd)(const DevPlan &, const void *A, void *packed, long long stride, int nb, long long pk_pitch, cudaStream_t);
    bool batch_fastest; // the launchers accept pk_pitch > 0
};
struct PlanTabs { ColTab ct; ColTab4 ct4; }; // column tables passed by value to the fast kernels
struct PlaneLaunch {
    int ry;
    int (*run[3])(const DevPlan &, const PlanTabs &, const void *Ain, void *Aout, const void *cin, void *cout, const void *v,
                  long long sin, long long sout, int nb, cudaStream_t);
    int nkern[3] = {1, 1, 1}; // kernels one run launches (the dense arm's plane stage is a y pass and an x pass)
};
// one cooperative launch per direction (fftb_fused.cuh): the intermediate lives in a ring of `nslot` band slots
struct FusedGeom { int ts, tile, rp; }; // sticks per z tile, elements of a tile's image, pitch of a row pair (ZFast)
struct FusedLaunch {
    FusedGeom geom;
    int (*inv)(const DevPlan &, const PlanTabs &, const void *packed, void *ring, const CUtensorMap &ring_map, void *cuboid, long long stride,
               int nb, int nslot, int lead, int nz, int hints, int *sync, cudaStream_t);
    int (*fwd)(const DevPlan &, const PlanTabs &, const void *cuboid, void *ring, void *packed, long long stride, int nb, int nslot,
               int lead, int nz, int hints, int *sync, cudaStream_t);
};

// cuTensorMapEncodeTiled through the runtime (no link against libcuda); looked up once
typedef CUresult (*tmap_encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *, const cuuint32_t *,
                                   const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
tmap_encode_fn tmap_encoder()
{
    static const tmap_encode_fn fn = [] {
        void *f = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &qres) != cudaSuccess || qres != cudaDriverEntryPointSuccess) {
            cudaGetLastError();
            f = nullptr;
        }
        return (tmap_encode_fn)f;
    }();
    return fn;
}
template <typename T, class AZ> int launch_zinv(const DevPlan &pl, const void *packed, void *A, long long stride, int nb, long long pk_pitch, cudaStream_t st)
{
    if (pk_pitch) return FFTB_EUNSUPPORTED;
    auto k = zpass_inv_k<T, AZ, Z_LINES, Z_NT>;
    const size_t smem = sizeof(cx<T>) * ((size_t)AZ::M * (Z_LINES | 1) + AZ::N);
    if (int rc = kernel_ready(k, Z_NT, smem, nullptr)) return rc;
    dim3 grid((pl.nsticks + Z_LINES - 1) / Z_LINES, nb);
    k<<<grid, Z_NT, smem, st>>>(pl, (const cx<T> *)packed, (cx<T> *)A, stride);
    return launch_status();
}
template <typename T, class AZ> int launch_zfwd(const DevPlan &pl, const void *A, void *packed, long long stride, int nb, long long pk_pitch, cudaStream_t st)
{
    if (pk_pitch) return FFTB_EUNSUPPORTED;
    auto k = zpass_fwd_k<T, AZ, Z_LINES, Z_NT>;
    const size_t smem = sizeof(cx<T>) * ((size_t)AZ::R * AZ::P2 * (AZ::P1 * (Z_LINES | 1) + 1) + AZ::N);
    if (int rc = kernel_ready(k, Z_NT, smem, nullptr)) return rc;
    dim3 grid((pl.nsticks + Z_LINES - 1) / Z_LINES, nb);
    k<<<grid, Z_NT, smem, st>>>(pl, (const cx<T> *)A, (cx<T> *)packed, stride);
    return launch_status();
}
template <typename T, class AX, class AY, int MODE>
int launch_plane(const DevPlan &pl, const PlanTabs &, const void *Ain, void *Aout, const void *cin, void *cout, const void *v, long long sin,
                 long long sout, int nb, cudaStream_t st)
{
    using TU = PlaneTune<AX, AY>;
    auto k = plane_k<T, AX, AY, TU::LX, TU::LY, TU::NT, MODE>;
    const size_t smem = PlaneSmem<T, AX, AY, TU::LX, TU::LY, TU::NT>::bytes;
    if (int rc = kernel_ready(k, TU::NT, smem, nullptr)) return rc;
    dim3 grid(AY::R * pl.n3, nb);
    k<<<grid, TU::NT, smem, st>>>(pl, (const cx<T> *)Ain, (cx<T> *)Aout, (const cx<T> *)cin, (cx<T> *)cout, (const T *)v, sin, sout);
    return launch_status();
}

// warp-synchronous persistent plane kernel (fftb_plane_fast.cuh): half-band power-of-two grids
constexpr int FAST_NW = 4; // warps per CTA of the z-pass kernels (4 CTAs per SM)
// warps per CTA of the plane kernel: a quarter of the x tasks of a plane
template <int N> struct PlaneNW { static constexpr int value = N >= 128 ? 8 : (N == 96 ? 4 : 2); }; // must divide N / G; measured best

template <typename T, class F, int MODE>
int launch_plane_fast(const DevPlan &pl, const PlanTabs &tabs, const void *Ain, void *Aout, const void *cin, void *cout, const void *v, long long sin,
                      long long sout, int nb, cudaStream_t st)
{
    constexpr int NW = PlaneNW<F::N>::value;
    auto k = plane_pf_k<T, F, NW, MODE>;
    const size_t smem = PlanePF<T, F, NW>::smem_bytes_mode(MODE, pl.pitch);
    if (smem > 227 * 1024) return FFTB_EUNSUPPORTED;
    int per_sm = 0;
    if (int rc = kernel_ready(k, NW * 32, smem, &per_sm)) return rc;
    const int nplanes = pl.n3 * nb;
    int grid = pl.sms * per_sm;
    if (grid > nplanes) grid = nplanes;
    k<<<grid, NW * 32, smem, st>>>(pl, tabs.ct, (const cx<T> *)Ain, (cx<T> *)Aout, (const cx<T> *)cin, (cx<T> *)cout, (const T *)v, sin, sout, nplanes);
    return launch_status();
}
template <typename T, int N, int P1, int P2> PlaneLaunch make_plane_fast()
{
    using F = FastCfg<T, N, P1, P2>;
    return PlaneLaunch{1, {&launch_plane_fast<T, F, MODE_INV>, &launch_plane_fast<T, F, MODE_FWD>, &launch_plane_fast<T, F, MODE_VLOC>}};
}
// The cuboids of a call as a tensor of real numbers for the TMA engine (256 pattern, fftb_plane_r4.cuh): an (x, x+1) pair | half of a group
// of four x | n' = x / 4 | y mod 4 | y / 4 over all planes and bands; a box = one half of the pairs of G = 4 lines four rows apart.
template <typename T> int r4_cuboid_map(CUtensorMap *cmap, const DevPlan &pl, const void *cuboid, int nb)
{
    const tmap_encode_fn enc = tmap_encoder();
    if (!enc) return FFTB_ECUDA;
    constexpr cuuint64_t E = sizeof(cx<T>), PAIR = 2 * E / sizeof(T);
    const cuuint64_t dims[5] = {PAIR, 2, 64, 4, (cuuint64_t)nb * pl.n3 * 64};
    const cuuint64_t strides[4] = {2 * E, 4 * E, 256 * E, 4 * 256 * E};
    const cuuint32_t box[5] = {(cuuint32_t)PAIR, 1, 64, 1, (cuuint32_t)PlaneR4<T, 8>::F::G};
    const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    if (enc(cmap, sizeof(T) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 5, const_cast<void *>(cuboid), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return FFTB_ECUDA;
    return 0;
}
// the 256 pattern parks per-thread values of the y tasks in tensor memory if every warp's y tasks fit its columns (fftb_plane_r4.cuh)
template <typename T> bool r4_tasks_fit_tmem(const DevPlan &pl)
{
    using R4 = PlaneR4<T, 8>;
    return ycol_tasks<typename R4::F>(pl.n_multi) <= R4::TMT * 8;
}
template <typename T, bool TM>
int launch_plane_r4_inv_tm(const DevPlan &pl, const PlanTabs &tabs, const void *Ain, void *cout, long long sin, int nb, cudaStream_t st)
{
    constexpr int NW = 8;
    auto k = plane_r4_inv_k<T, NW, TM>;
    const size_t smem = PlaneR4<T, NW>::smem_bytes;
    if (int rc = kernel_ready(k, NW * 32, smem, nullptr)) return rc;
    const int nplanes = pl.n3 * nb;
    int grid = pl.sms;
    if (grid > nplanes) grid = nplanes;
    CUtensorMap cmap;
    if (int rc = r4_cuboid_map<T>(&cmap, pl, cout, nb)) return rc;
    k<<<grid, NW * 32, smem, st>>>(pl, tabs.ct4, (const cx<T> *)Ain, (cx<T> *)cout, cmap, sin, nplanes);
    return launch_status();
}
// inverse plane kernel of the 256 pattern (fftb_plane_r4.cuh)
template <typename T>
int launch_plane_r4_inv(const DevPlan &pl, const PlanTabs &tabs, const void *Ain, void *, const void *, void *cout, const void *, long long sin,
                        long long, int nb, cudaStream_t st)
{
    return r4_tasks_fit_tmem<T>(pl) ? launch_plane_r4_inv_tm<T, true>(pl, tabs, Ain, cout, sin, nb, st)
                                    : launch_plane_r4_inv_tm<T, false>(pl, tabs, Ain, cout, sin, nb, st);
}

template <typename T, bool TM>
int launch_plane_r4_vloc_tm(const DevPlan &pl, const PlanTabs &tabs, const void *Ain, void *Aout, const void *v, long long sin, long long sout, int nb,
                            cudaStream_t st)
{
    constexpr int NW = 8;
    auto k = plane_r4_vloc_k<T, NW, TM>;
    const size_t smem = PlaneR4<T, NW>::smem_bytes;
    if (int rc = kernel_ready(k, NW * 32, smem, nullptr)) return rc;
    const int nplanes = pl.n3 * nb;
    int grid = pl.sms;
    if (grid > nplanes) grid = nplanes;
    k<<<grid, NW * 32, smem, st>>>(pl, tabs.ct4, (const cx<T> *)Ain, (cx<T> *)Aout, (const T *)v, sin, sout, nplanes);
    return launch_status();
}
template <typename T>
int launch_plane_r4_vloc(const DevPlan &pl, const PlanTabs &tabs, const void *Ain, void *Aout, const void *, void *, const void *v, long long sin,
                         long long sout, int nb, cudaStream_t st)
{
    return r4_tasks_fit_tmem<T>(pl) ? launch_plane_r4_vloc_tm<T, true>(pl, tabs, Ain, Aout, v, sin, sout, nb, st)
                                    : launch_plane_r4_vloc_tm<T, false>(pl, tabs, Ain, Aout, v, sin, sout, nb, st);
}

template <typename T, bool TM>
int launch_plane_r4_fwd_tm(const DevPlan &pl, const PlanTabs &tabs, const void *cin, void *Aout, long long sout, int nb, cudaStream_t st)
{
    constexpr int NW = 8;
    using R4 = PlaneR4<T, NW>;
    auto k = plane_r4_fwd_k<T, NW, TM>;
    const size_t smem = R4::smem_bytes_fwd;
    if (int rc = kernel_ready(k, NW * 32, smem, nullptr)) return rc;
    CUtensorMap cmap;
    if (int rc = r4_cuboid_map<T>(&cmap, pl, cin, nb)) return rc;
    const int nplanes = pl.n3 * nb;
    int grid = pl.sms;
    if (grid > nplanes) grid = nplanes;
    k<<<grid, NW * 32, smem, st>>>(pl, tabs.ct4, cmap, (cx<T> *)Aout, sout, nplanes);
    return launch_status();
}
template <typename T>
int launch_plane_r4_fwd(const DevPlan &pl, const PlanTabs &tabs, const void *, void *Aout, const void *cin, void *, const void *, long long,
                        long long sout, int nb, cudaStream_t st)
{
    return r4_tasks_fit_tmem<T>(pl) ? launch_plane_r4_fwd_tm<T, true>(pl, tabs, cin, Aout, sout, nb, st)
                                   : launch_plane_r4_fwd_tm<T, false>(pl, tabs, cin, Aout, sout, nb, st);
}

bool find_plane_fast(int dtype, int n, bool dense, PlaneLaunch *out)
{
    if (dense) return false;
    if (dtype == FFTB_C128 && n == 128) { *out = make_plane_fast<double, 128, 8, 8>(); return true; }
    if (dtype == FFTB_C128 && n == 64) { *out = make_plane_fast<double, 64, 8, 4>(); return true; }
    if (dtype == FFTB_C64 && n == 128) { *out = make_plane_fast<float, 128, 8, 8>(); return true; }
    if (dtype == FFTB_C64 && n == 64) { *out = make_plane_fast<float, 64, 8, 4>(); return true; }
    if (dtype == FFTB_C64 && n == 96) { *out = make_plane_fast<float, 96, 12, 4>(); return true; }   // 48 = 12 x 4
    if (dtype == FFTB_C128 && n == 96) { *out = make_plane_fast<double, 96, 12, 4>(); return true; }
    return false;
}

// persistent z-pass kernels: grid = resident CTAs (shared memory decides: 3 per SM at N3 = 64, 128; 2 at 96), tiles strided over it
template <class K> int zpers_launch_grid(K kp, int threads, size_t smem, const DevPlan &pl, int total, int *grid)
{
    int per_sm = 0;
    if (int rc = kernel_ready(kp, threads, smem, &per_sm)) return rc;
    const int cap = pl.sms * per_sm;
    *grid = total < cap ? total : cap;
    return 0;
}

// The intermediate of a z-pass launch as a tensor of real numbers for the TMA engine (fftb_zpass_pf.cuh): reals of a row of A | (z / 2) mod 8 |
// z / 16 | z mod 2 | band; a box = the 128 bytes of SG sticks x all N3 rows of one band (in that order), written / read with the 128-byte swizzle.
template <typename T> int z_a_map(CUtensorMap *amap, const DevPlan &pl, const void *A, long long stride, int nb)
{
    const tmap_encode_fn enc = tmap_encoder();
    if (!enc) return FFTB_ECUDA;
    constexpr cuuint64_t E = sizeof(cx<T>);
    const cuuint64_t row = (cuuint64_t)pl.pitch * E;
    const cuuint64_t dims[5] = {(cuuint64_t)pl.pitch * (E / sizeof(T)), 8, (cuuint64_t)pl.n3 / 16, 2, (cuuint64_t)nb};
    const cuuint64_t strides[4] = {2 * row, 16 * row, row, (cuuint64_t)(stride > 0 ? stride : (long long)pl.n3 * pl.pitch) * E};
    const cuuint32_t box[5] = {(cuuint32_t)(128 / sizeof(T)), 8, (cuuint32_t)(pl.n3 / 16), 2, 1};
    const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    if (pl.n3 % 16) return FFTB_EUNSUPPORTED;
    if (enc(amap, sizeof(T) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 5, const_cast<void *>(A), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return FFTB_ECUDA;
    return 0;
}
template <typename T, class F> int launch_zfast_inv(const DevPlan &pl, const void *packed, void *A, long long stride, int nb, long long pk_pitch, cudaStream_t st)
{
    // persistent kernel, global memory moved by the TMA engine only (batch-fastest packed arrays: per-element cp.async)
    const int ntiles = (pl.nsticks + F::G * FAST_NW - 1) / (F::G * FAST_NW), total = ntiles * nb;
    using ZP = ZPers<T, F, FAST_NW>;
    auto kp = pk_pitch ? zpass_pers_inv_k<T, F, FAST_NW, true> : zpass_pers_inv_k<T, F, FAST_NW, false>;
    int grid = 0;
    if (int rc = zpers_launch_grid(kp, FAST_NW * 32, ZP::smem_bytes, pl, total, &grid)) return rc;
    CUtensorMap amap;
    if (int rc = z_a_map<T>(&amap, pl, A, stride, nb)) return rc;
    kp<<<grid, FAST_NW * 32, ZP::smem_bytes, st>>>(pl, (const cx<T> *)packed, amap, ntiles, total, pk_pitch);
    return launch_status();
}
template <typename T, class F> int launch_zfast_fwd(const DevPlan &pl, const void *A, void *packed, long long stride, int nb, long long pk_pitch, cudaStream_t st)
{
    const int ntiles = (pl.nsticks + F::G * FAST_NW - 1) / (F::G * FAST_NW), total = ntiles * nb;
    if (pl.ry == 1) { // one plane of A (fast plane kernels): persistent kernel
        using ZP = ZPers<T, F, FAST_NW>;
        auto kp = pk_pitch ? zpass_pers_fwd_k<T, F, FAST_NW, true> : zpass_pers_fwd_k<T, F, FAST_NW, false>;
        int grid = 0;
        if (int rc = zpers_launch_grid(kp, FAST_NW * 32, ZP::smem_bytes, pl, total, &grid)) return rc;
        CUtensorMap amap;
        if (int rc = z_a_map<T>(&amap, pl, A, stride, nb)) return rc;
        kp<<<grid, FAST_NW * 32, ZP::smem_bytes, st>>>(pl, amap, (cx<T> *)packed, ntiles, total, pk_pitch);
        return launch_status();
    }
    if (pk_pitch) return FFTB_EUNSUPPORTED;
    auto k = zpass_fast_fwd_k<T, F, FAST_NW>; // partial planes of the generic plane kernel are summed here
    const size_t smem = ZFast<T, F, FAST_NW>::smem_bytes;
    if (int rc = kernel_ready(k, FAST_NW * 32, smem, nullptr)) return rc;
    k<<<dim3(ntiles, nb), FAST_NW * 32, smem, st>>>(pl, (const cx<T> *)A, (cx<T> *)packed, stride);
    return launch_status();
}
template <typename T, int N, int P1, int P2> ZLaunch make_z_fast()
{
    using F = FastCfg<T, N, P1, P2>;
    return ZLaunch{&launch_zfast_inv<T, F>, &launch_zfast_fwd<T, F>, true};
}
// z passes of the 256 pattern (fftb_plane_r4.cuh)
constexpr int R4Z_NW = 4;
// The intermediate of a z-pass launch as a tensor of real numbers for the TMA engine (fftb_zpass_pf.cuh): reals of a row of A | n' mod 8 | n' / 8 |
// z mod 4 | band (z = 4 n' + e); a box = the 128 bytes of SG sticks x all 64 n' x 2 consecutive residues of one band, written / read with the 128-byte swizzle.
template <typename T> int zr4_a_map(CUtensorMap *amap, const DevPlan &pl, const void *A, long long stride, int nb)
{
    const tmap_encode_fn enc = tmap_encoder();
    if (!enc) return FFTB_ECUDA;
    constexpr cuuint64_t E = sizeof(cx<T>);
    const cuuint64_t row = (cuuint64_t)pl.pitch * E;
    const cuuint64_t dims[5] = {(cuuint64_t)pl.pitch * (E / sizeof(T)), 8, 8, 4, (cuuint64_t)nb};
    const cuuint64_t strides[4] = {4 * row, 32 * row, row, (cuuint64_t)(stride > 0 ? stride : (long long)pl.n3 * pl.pitch) * E};
    const cuuint32_t box[5] = {(cuuint32_t)(128 / sizeof(T)), 8, 8, 2, 1};
    const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    if (enc(amap, sizeof(T) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 5, const_cast<void *>(A), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return FFTB_ECUDA;
    return 0;
}
template <typename T> int launch_zr4_inv(const DevPlan &pl, const void *packed, void *A, long long stride, int nb, long long pk_pitch, cudaStream_t st)
{
    if (pk_pitch) return FFTB_EUNSUPPORTED;
    using ZP = ZPersR4<T, R4Z_NW>;
    auto kp = zpass_r4_pers_inv_k<T, R4Z_NW>;
    const int ntiles = (pl.nsticks + ZP::TS - 1) / ZP::TS, total = ntiles * nb;
    int grid = 0;
    if (int rc = zpers_launch_grid(kp, R4Z_NW * 32, ZP::smem_bytes, pl, total, &grid)) return rc;
    CUtensorMap amap;
    if (int rc = zr4_a_map<T>(&amap, pl, A, stride, nb)) return rc;
    kp<<<grid, R4Z_NW * 32, ZP::smem_bytes, st>>>(pl, (const cx<T> *)packed, amap, ntiles, total);
    return launch_status();
}
template <typename T> int launch_zr4_fwd(const DevPlan &pl, const void *A, void *packed, long long stride, int nb, long long pk_pitch, cudaStream_t st)
{
    if (pk_pitch) return FFTB_EUNSUPPORTED;
    if (pl.ry == 1) { // one plane of A (the 256 pattern's own plane kernels): persistent kernel
        using ZP = ZPersR4<T, R4Z_NW>;
        auto kp = zpass_r4_pers_fwd_k<T, R4Z_NW>;
        const int ntiles = (pl.nsticks + ZP::TS - 1) / ZP::TS, total = ntiles * nb;
        int grid = 0;
        if (int rc = zpers_launch_grid(kp, R4Z_NW * 32, ZP::smem_bytes, pl, total, &grid)) return rc;
        CUtensorMap amap;
        if (int rc = zr4_a_map<T>(&amap, pl, A, stride, nb)) return rc;
        kp<<<grid, R4Z_NW * 32, ZP::smem_bytes, st>>>(pl, amap, (cx<T> *)packed, ntiles, total);
        return launch_status();
    }
    auto k = zpass_r4_fwd_k<T, R4Z_NW>;
    const size_t smem = ZR4<T, R4Z_NW>::smem_bytes;
    if (int rc = kernel_ready(k, R4Z_NW * 32, smem, nullptr)) return rc;
    dim3 grid((pl.nsticks + ZR4<T, R4Z_NW>::TS - 1) / ZR4<T, R4Z_NW>::TS, nb);
    k<<<grid, R4Z_NW * 32, smem, st>>>(pl, (const cx<T> *)A, (cx<T> *)packed, stride);
    return launch_status();
}

bool find_z_fast(int dtype, int n, bool dense, ZLaunch *out)
{
    if (dense) return false;
    if (dtype == FFTB_C128 && n == 256) { *out = ZLaunch{&launch_zr4_inv<double>, &launch_zr4_fwd<double>, false}; return true; }
    if (dtype == FFTB_C64 && n == 256) { *out = ZLaunch{&launch_zr4_inv<float>, &launch_zr4_fwd<float>, false}; return true; }
    if (dtype == FFTB_C128 && n == 128) { *out = make_z_fast<double, 128, 8, 8>(); return true; }
    if (dtype == FFTB_C128 && n == 64) { *out = make_z_fast<double, 64, 8, 4>(); return true; }
    if (dtype == FFTB_C64 && n == 128) { *out = make_z_fast<float, 128, 8, 8>(); return true; }
    if (dtype == FFTB_C64 && n == 64) { *out = make_z_fast<float, 64, 8, 4>(); return true; }
    if (dtype == FFTB_C64 && n == 96) { *out = make_z_fast<float, 96, 12, 4>(); return true; }
    if (dtype == FFTB_C128 && n == 96) { *out = make_z_fast<double, 96, 12, 4>(); return true; }
    if (dtype == FFTB_C64 && n == 192) { *out = make_z_fast<float, 192, 24, 4>(); return true; }     // 96 = 24 x 4
    return false;
}

// ------------------------------------------------------------------------------------------------
// fused launches (fftb_fused.cuh): cubic grids whose z axis uses the plane kernel's factorisation
// ------------------------------------------------------------------------------------------------
template <class K> int fused_grid(K k, int threads, size_t smem, const DevPlan &pl, int items, int *grid)
{
    int per_sm = 0;
    if (int rc = kernel_ready(k, threads, smem, &per_sm)) return rc;
    const int cap = pl.sms * per_sm; // every CTA of a cooperative launch is resident
    *grid = items < cap ? items : cap;
    return 0;
}
template <typename T, class F>
int launch_fused_inv(const DevPlan &pl, const PlanTabs &tabs, const void *packed, void *ring, const CUtensorMap &ring_map, void *cuboid,
                     long long stride, int nb, int nslot, int lead, int nz, int hints, int *sync, cudaStream_t st)
{
    constexpr int NW = PlaneNW<F::N>::value;
    using FU = Fused<T, F, NW>;
    auto k = fused_inv_k<T, F, NW>;
    const int ntiles = (pl.nsticks + FU::Z::TS - 1) / FU::Z::TS;
    const size_t smem = FU::smem_inv(ntiles);
    if (smem > 227 * 1024) return FFTB_EUNSUPPORTED;
    const int items = nb * (pl.n3 > ntiles ? pl.n3 : ntiles);
    int grid = 0;
    if (int rc = fused_grid(k, NW * 32, smem, pl, items, &grid)) return rc;
    if (nz >= grid) nz = 0; // spatial split needs CTAs of both roles: fall back to the merged walk
    if (cudaMemsetAsync(sync, 0, 2 * sizeof(int) * (size_t)nb, st) != cudaSuccess) return FFTB_ECUDA;
    const cx<T> *a_packed = (const cx<T> *)packed;
    cx<T> *a_ring = (cx<T> *)ring, *a_cub = (cx<T> *)cuboid;
    int *zdone = sync, *pdone = sync + nb;
    void *args[] = {(void *)&pl, (void *)&tabs.ct, (void *)&a_packed, (void *)&a_ring, (void *)&ring_map, (void *)&a_cub, (void *)&stride,
                    (void *)&nb, (void *)&nslot, (void *)&lead, (void *)&nz, (void *)&hints, (void *)&zdone, (void *)&pdone};
    if (cudaLaunchCooperativeKernel((const void *)k, dim3(grid), dim3(NW * 32), args, smem, st) != cudaSuccess) return FFTB_ECUDA;
    return launch_status();
}
template <typename T, class F>
int launch_fused_fwd(const DevPlan &pl, const PlanTabs &tabs, const void *cuboid, void *ring, void *packed, long long stride, int nb, int nslot,
                     int lead, int nz, int hints, int *sync, cudaStream_t st)
{
    constexpr int NW = PlaneNW<F::N>::value;
    using FU = Fused<T, F, NW>;
    auto k = fused_fwd_k<T, F, NW>;
    const size_t smem = FU::smem_fwd;
    const int ntiles = (pl.nsticks + FU::Z::TS - 1) / FU::Z::TS;
    const int items = nb * (pl.n3 > ntiles ? pl.n3 : ntiles);
    int grid = 0;
    if (int rc = fused_grid(k, NW * 32, smem, pl, items, &grid)) return rc;
    if (nz >= grid) nz = 0;
    if (cudaMemsetAsync(sync, 0, 2 * sizeof(int) * (size_t)nb, st) != cudaSuccess) return FFTB_ECUDA;
    const cx<T> *a_cub = (const cx<T> *)cuboid;
    cx<T> *a_ring = (cx<T> *)ring, *a_packed = (cx<T> *)packed;
    int *pdone = sync, *zdone = sync + nb;
    void *args[] = {(void *)&pl, (void *)&tabs.ct, (void *)&a_cub, (void *)&a_ring, (void *)&a_packed, (void *)&stride, (void *)&nb,
                    (void *)&nslot, (void *)&lead, (void *)&nz, (void *)&hints, (void *)&pdone, (void *)&zdone};
    if (cudaLaunchCooperativeKernel((const void *)k, dim3(grid), dim3(NW * 32), args, smem, st) != cudaSuccess) return FFTB_ECUDA;
    return launch_status();
}
template <typename T, int N, int P1, int P2> FusedLaunch make_fused()
{
    using F = FastCfg<T, N, P1, P2>;
    static_assert(Fused<T, F, PlaneNW<N>::value>::smem_fwd <= 227 * 1024, "fused forward kernel does not fit in shared memory");
    using Z = typename Fused<T, F, PlaneNW<N>::value>::Z;
    return FusedLaunch{FusedGeom{Z::TS, Z::TILE, Z::RP}, &launch_fused_inv<T, F>, &launch_fused_fwd<T, F>};
}
bool find_fused(int dtype, const int32_t n[3], bool dense, FusedLaunch *out)
{
    if (dense || n[0] != n[1] || n[0] != n[2]) return false;
    if (dtype == FFTB_C128 && n[0] == 128) { *out = make_fused<double, 128, 8, 8>(); return true; }
    if (dtype == FFTB_C64 && n[0] == 128) { *out = make_fused<float, 128, 8, 8>(); return true; }
    return false;
}

// ------------------------------------------------------------------------------------------------
// dense arm (fftb_dense.cuh): three line passes per direction on the warp-synchronous core, cubic grids
// ------------------------------------------------------------------------------------------------
constexpr int DENSE_NW = 4;
template <typename T, class F, int MODE, bool PAIR>
int launch_dense_axis(const void *in, void *out, const DenseGeom &ge, const void *tw, const void *v, double scale, int nb, cudaStream_t st)
{
    auto k = dense_axis_k<T, F, DENSE_NW, MODE, PAIR>;
    const size_t smem = sizeof(cx<T>) * (size_t)DENSE_NW * F::EXW;
    if (int rc = kernel_ready(k, DENSE_NW * 32, smem, nullptr)) return rc;
    constexpr int per_cta = DENSE_NW * F::G;
    dim3 grid((ge.lines + per_cta - 1) / per_cta, nb);
    k<<<grid, DENSE_NW * 32, smem, st>>>((const cx<T> *)in, (cx<T> *)out, ge, (const cx<T> *)tw, (const T *)v, (T)scale);
    return launch_status();
}
// the passes as strides; A[z][k1][k2] with row pitch pl.pitch = N1 N2 (the dense stick map: stick s = k1 N2 + k2)
inline DenseGeom dense_geom_z(const DevPlan &pl, long long a_stride, bool inverse)
{
    // packed [stick][k3] <-> A[z][stick]
    DenseGeom p2a = {0, pl.n3, 1, 0, 1, pl.pitch, pl.S, a_stride, pl.nsticks, pl.nsticks};
    DenseGeom a2p = {0, 1, pl.pitch, 0, pl.n3, 1, a_stride, pl.S, pl.nsticks, pl.nsticks};
    return inverse ? p2a : a2p;
}
inline DenseGeom dense_geom_y(const DevPlan &pl, long long a_stride)
{
    // in place on A: line (z, k1) is contiguous in k2 / y
    return DenseGeom{pl.pitch, pl.n2, 1, pl.pitch, pl.n2, 1, a_stride, a_stride, pl.n1, pl.n3 * pl.n1};
}
inline DenseGeom dense_geom_x(const DevPlan &pl, long long a_in, long long a_out, int side) // 0: A -> cuboid, 1: cuboid -> A, 2: A -> A
{
    const long long C = (long long)pl.n1 * pl.n2 * pl.n3, row = pl.n1, plane = (long long)pl.n1 * pl.n2;
    DenseGeom g;
    g.nv = pl.n2;
    g.lines = pl.n3 * pl.n2;
    if (side == 1) { g.in_u = plane; g.in_v = row; g.in_i = 1; g.in_band = C; }
    else { g.in_u = pl.pitch; g.in_v = 1; g.in_i = pl.n2; g.in_band = a_in; }
    if (side == 0) { g.out_u = plane; g.out_v = row; g.out_i = 1; g.out_band = C; }
    else { g.out_u = pl.pitch; g.out_v = 1; g.out_i = pl.n2; g.out_band = a_out; }
    return g;
}
template <typename T, class F> int launch_dense_zinv(const DevPlan &pl, const void *packed, void *A, long long stride, int nb, long long pk_pitch, cudaStream_t st)
{
    if (pk_pitch) return FFTB_EUNSUPPORTED;
    return launch_dense_axis<T, F, DENSE_INV, false>(packed, A, dense_geom_z(pl, stride, true), pl.tw3, nullptr, 1.0, nb, st);
}
template <typename T, class F> int launch_dense_zfwd(const DevPlan &pl, const void *A, void *packed, long long stride, int nb, long long pk_pitch, cudaStream_t st)
{
    if (pk_pitch) return FFTB_EUNSUPPORTED;
    return launch_dense_axis<T, F, DENSE_FWD, false>(A, packed, dense_geom_z(pl, stride, false), pl.tw3, nullptr, pl.scale, nb, st);
}
template <typename T, class F>
int launch_dense_plane_inv(const DevPlan &pl, const PlanTabs &, const void *Ain, void *, const void *, void *cout, const void *, long long sin, long long,
                           int nb, cudaStream_t st)
{
    void *A = const_cast<void *>(Ain); // the workspace: the y pass works on it in place
    if (int rc = launch_dense_axis<T, F, DENSE_INV, true>(A, A, dense_geom_y(pl, sin), pl.tw2, nullptr, 1.0, nb, st)) return rc;
    return launch_dense_axis<T, F, DENSE_INV, true>(A, cout, dense_geom_x(pl, sin, 0, 0), pl.tw1, nullptr, 1.0, nb, st);
}
template <typename T, class F>
int launch_dense_plane_fwd(const DevPlan &pl, const PlanTabs &, const void *, void *Aout, const void *cin, void *, const void *, long long, long long sout,
                           int nb, cudaStream_t st)
{
    if (int rc = launch_dense_axis<T, F, DENSE_FWD, true>(cin, Aout, dense_geom_x(pl, 0, sout, 1), pl.tw1, nullptr, 1.0, nb, st)) return rc;
    return launch_dense_axis<T, F, DENSE_FWD, true>(Aout, Aout, dense_geom_y(pl, sout), pl.tw2, nullptr, 1.0, nb, st);
}
template <typename T, class F>
int launch_dense_plane_vloc(const DevPlan &pl, const PlanTabs &, const void *Ain, void *Aout, const void *, void *, const void *v, long long sin,
                            long long sout, int nb, cudaStream_t st)
{
    void *A = const_cast<void *>(Ain);
    if (int rc = launch_dense_axis<T, F, DENSE_INV, true>(A, A, dense_geom_y(pl, sin), pl.tw2, nullptr, 1.0, nb, st)) return rc;
    if (int rc = launch_dense_axis<T, F, DENSE_VLOC, true>(A, Aout, dense_geom_x(pl, sin, sout, 2), pl.tw1, v, 1.0, nb, st)) return rc;
    return launch_dense_axis<T, F, DENSE_FWD, true>(Aout, Aout, dense_geom_y(pl, sout), pl.tw2, nullptr, 1.0, nb, st);
}
template <typename T, int N, int P1, int P2> void make_dense_fast(ZLaunch *zl, PlaneLaunch *plk)
{
    using F = FastCfg<T, N, P1, P2>;
    *zl = ZLaunch{&launch_dense_zinv<T, F>, &launch_dense_zfwd<T, F>, false};
    *plk = PlaneLaunch{1, {&launch_dense_plane_inv<T, F>, &launch_dense_plane_fwd<T, F>, &launch_dense_plane_vloc<T, F>}, {2, 2, 3}};
}
bool find_dense_fast(int dtype, const int32_t n[3], ZLaunch *zl, PlaneLaunch *plk)
{
    if (n[0] != n[1] || n[0] != n[2]) return false;
#define DCASE(N, P1, P2) \
    if (n[0] == N) { if (dtype == FFTB_C128) make_dense_fast<double, N, P1, P2>(zl, plk); else make_dense_fast<float, N, P1, P2>(zl, plk); return true; }
    DCASE(64, 8, 4) DCASE(128, 8, 8) DCASE(256, 16, 8)
#undef DCASE
    return false;
}

template <typename T, int N, bool DENSE> ZLaunch make_z()
{
    using AZ = typename ZX<N, DENSE>::type;
    return ZLaunch{&launch_zinv<T, AZ>, &launch_zfwd<T, AZ>, false};
}
template <typename T, int N, bool DENSE> PlaneLaunch make_plane()
{
    using AX = typename ZX<N, DENSE>::type;
    using AY = typename YA<N, DENSE>::type;
    static_assert(PlaneSmem<T, AX, AY, PlaneTune<AX, AY>::LX, PlaneTune<AX, AY>::LY, PlaneTune<AX, AY>::NT>::bytes <= 227 * 1024,
                  "plane does not fit in shared memory");
    return PlaneLaunch{AY::R,
                       {&launch_plane<T, AX, AY, MODE_INV>, &launch_plane<T, AX, AY, MODE_FWD>, &launch_plane<T, AX, AY, MODE_VLOC>}};
}

// rectangular x/y grids (N1 != N2): the generic plane kernel with one axis pattern per axis
template <typename T, int NX, int NY> PlaneLaunch make_plane_xy()
{
    using AX = typename ZX<NX, false>::type;
    using AY = typename YA<NY, false>::type;
    static_assert(PlaneSmem<T, AX, AY, PlaneTune<AX, AY>::LX, PlaneTune<AX, AY>::LY, PlaneTune<AX, AY>::NT>::bytes <= 227 * 1024,
                  "plane does not fit in shared memory");
    return PlaneLaunch{AY::R,
                       {&launch_plane<T, AX, AY, MODE_INV>, &launch_plane<T, AX, AY, MODE_FWD>, &launch_plane<T, AX, AY, MODE_VLOC>}};
}
bool find_plane_xy(int dtype, int nx, int ny, PlaneLaunch *out)
{
#define XYCASE(NX, NY) \
    if (nx == NX && ny == NY) { *out = dtype == FFTB_C128 ? make_plane_xy<double, NX, NY>() : make_plane_xy<float, NX, NY>(); return true; }
    XYCASE(32, 64) XYCASE(64, 32) XYCASE(64, 128) XYCASE(128, 64)
#undef XYCASE
    return false;
}

bool find_z(int dtype, int n, bool dense, ZLaunch *out)
{
#define ZCASE(T, DT, N, D) \
    if (dtype == DT && n == N && dense == D) { *out = make_z<T, N, D>(); return true; }
    ZCASE(double, FFTB_C128, 32, false) ZCASE(double, FFTB_C128, 64, false) ZCASE(double, FFTB_C128, 96, false)
    ZCASE(double, FFTB_C128, 128, false) ZCASE(double, FFTB_C128, 192, false) ZCASE(double, FFTB_C128, 256, false)
    ZCASE(float, FFTB_C64, 32, false) ZCASE(float, FFTB_C64, 64, false) ZCASE(float, FFTB_C64, 96, false)
    ZCASE(float, FFTB_C64, 128, false) ZCASE(float, FFTB_C64, 192, false) ZCASE(float, FFTB_C64, 256, false)
    ZCASE(double, FFTB_C128, 32, true) ZCASE(double, FFTB_C128, 64, true) ZCASE(double, FFTB_C128, 128, true)
    ZCASE(double, FFTB_C128, 256, true)
    ZCASE(float, FFTB_C64, 32, true) ZCASE(float, FFTB_C64, 64, true) ZCASE(float, FFTB_C64, 128, true) ZCASE(float, FFTB_C64, 256, true)
#undef ZCASE
    return false;
}
bool find_plane(int dtype, int n, bool dense, PlaneLaunch *out)
{
#define PCASE(T, DT, N, D) \
    if (dtype == DT && n == N && dense == D) { *out = make_plane<T, N, D>(); return true; }
    PCASE(double, FFTB_C128, 32, false) PCASE(double, FFTB_C128, 64, false) PCASE(double, FFTB_C128, 96, false)
    PCASE(double, FFTB_C128, 128, false) PCASE(double, FFTB_C128, 192, false) PCASE(double, FFTB_C128, 256, false)
    PCASE(float, FFTB_C64, 32, false) PCASE(float, FFTB_C64, 64, false) PCASE(float, FFTB_C64, 96, false)
    PCASE(float, FFTB_C64, 128, false) PCASE(float, FFTB_C64, 192, false) PCASE(float, FFTB_C64, 256, false)
    PCASE(double, FFTB_C128, 32, true) PCASE(double, FFTB_C128, 64, true) PCASE(double, FFTB_C128, 128, true)
    PCASE(double, FFTB_C128, 256, true)
    PCASE(float, FFTB_C64, 32, true) PCASE(float, FFTB_C64, 64, true) PCASE(float, FFTB_C64, 128, true) PCASE(float, FFTB_C64, 256, true)
#undef PCASE
    return false;
}

// ------------------------------------------------------------------------------------------------
// cut-off membership in exact integers (Eq. 9, inclusive)
// ------------------------------------------------------------------------------------------------
bool inside(long long k1, long long k2, long long k3, const int32_t a[3])
{
    long long w[3];
    const long long k[3] = {k1, k2, k3};
    for (int d = 0; d < 3; ++d) {
        if (a[d] == 0 && k[d] != 0) return false;
        w[d] = a[d] ? a[d] : 1;
    }
    const long long lhs = k1 * k1 * (w[1] * w[2]) * (w[1] * w[2]) + k2 * k2 * (w[0] * w[2]) * (w[0] * w[2]) +
                          k3 * k3 * (w[0] * w[1]) * (w[0] * w[1]);
    return lhs <= (w[0] * w[1] * w[2]) * (w[0] * w[1] * w[2]);
}

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

} // namespace

struct fftb_plan_s {
    fftb_plan_desc desc;
    bool dense;
    size_t elem;
    int64_t S, C;
    int nsticks, nxocc, pitch, k1lo, ry;
    int nphantom; // zero-length sticks the builder put into the holes of an explicit map (counted in nsticks, hidden from the caller)
    std::vector<int32_t> k1, k2, k3lo, len;
    std::vector<int64_t> off;
    std::vector<int4> h_stick, h_col;
    std::vector<int> h_colperm;
    int n_multi;
    std::vector<unsigned char> h_tw[3];
    ZLaunch zl;
    PlaneLaunch plk;
    FusedLaunch ful;
    bool fused;          // fftb_inverse / fftb_forward are ONE cooperative launch each (fftb_fused.cuh)
    bool bf;             // packed arrays are batch-fastest: [point][band], nb bands per point in a call with nb bands
    int ring_bands, lead_bands; // the fused kernels' ring of intermediate band slots and the producers' lead
    int l2_hints;        // fused kernels: evict_last on the ring, evict_first on the cuboid and packed streams
    int z_ctas;          // fused kernels: > 0 = spatial split, this many CTAs walk the z tiles only (fftb_fused.cuh)
    long long ring_slot; // elements of a ring slot: ntiles tile images (tile-major layout, fftb_fused.cuh)
    int ring_ntiles;
    CUtensorMap ring_map; // the ring as a 5-dimensional tensor (inverse plane items load a row out of every tile)
    // device block layout
    size_t o_stick, o_col, o_perm, o_tw[3], o_sync, o_ws, o_stage[2], o_stage_out[2], bytes_min, bytes_stage;
    long long a_inv_stride, a_fwd_stride; // elements per band of the intermediate (a_fwd_stride: vloc and generic forward)
    int chunk;                            // bands per kernel group (vloc: both intermediates live)
    int chunk_inv, chunk_fwd;             // inverse / forward alone
    // bound state
    unsigned char *d_mem;
    bool staging;
    // *_host calls: the packed arrays cross PCIe in HOST_PIPE band chunks on two private copy streams, so
    // that a chunk's copy runs while its neighbours are transformed (created once in fftb_plan_bind)
    cudaStream_t cs_in, cs_out;
    cudaEvent_t hev_in_free[2], hev_done[2], hev_in[8], hev_out[8];
    bool in_free_recorded[2], done_recorded[2]; // the event has been recorded at least once
    // FFTB_TUNE_HOST_DEFER: two incoming and two outgoing staging areas, taken in turn by successive *_host calls, and no
    // wait of the caller's stream for a call's device-to-host copies (fftb_host_flush does that)
    bool host_defer;
    unsigned host_in_calls, host_out_calls;
    bool pipe_ok;
    DevPlan dev;
    PlanTabs tabs; // the column table again, as a by-value kernel parameter of the fast plane kernels
    int sticky;
    int launches;
    // optional per-kernel timing (fftb_plan_profile): event pairs recorded around every launch
    bool prof;
    std::vector<cudaEvent_t> ev;   // pairs
    std::vector<int> ev_kind;      // kernel kind of each pair
    size_t ev_used;
};

enum { K_ZINV = 0, K_PLANE_INV = 1, K_PLANE_FWD = 2, K_ZFWD = 3, K_PLANE_VLOC = 4, K_FUSED_INV = 5, K_FUSED_FWD = 6, K_KINDS = 7 };

static void prof_begin(fftb_plan p, int kind, cudaStream_t st)
{
    if (!p->prof) return;
    if (p->ev_used + 2 > p->ev.size()) {
        cudaEvent_t a, b;
        if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) { p->prof = false; return; }
        p->ev.push_back(a);
        p->ev.push_back(b);
        p->ev_kind.push_back(kind);
    }
    p->ev_kind[p->ev_used / 2] = kind;
    cudaEventRecord(p->ev[p->ev_used], st);
}
static void prof_end(fftb_plan p, cudaStream_t st)
{
    if (!p->prof) return;
    cudaEventRecord(p->ev[p->ev_used + 1], st);
    p->ev_used += 2;
}

extern "C" {

const char *fftb_strerror(int code)
{
    switch (code) {
    case FFTB_OK: return "ok";
    case FFTB_EINVAL: return "invalid argument";
    case FFTB_EUNSUPPORTED: return "description outside the predefined patterns";
    case FFTB_ENOMEM: return "out of memory / bind block too small";
    case FFTB_ECUDA: return "CUDA error";
    case FFTB_ESTATE: return "plan not bound / mismatched plans";
    case FFTB_ETOOBIG: return "transform too large for the static scratch array (FFTB_STATIC_SCRATCH_BYTES)";
    default: return "unknown fftb status";
    }
}

struct ExplicitMap { int64_t n; const int32_t *k1, *k2, *k3lo, *len; };

static int plan_create_impl(fftb_plan *out, const fftb_plan_desc *desc, const ExplicitMap *xm, const fftb_plan_tuning *tune)
{
    if (!out || !desc) return FFTB_EINVAL;
    *out = nullptr;
    const uint32_t tflags = tune ? tune->flags : 0u;
    if (tflags & ~(uint32_t)(FFTB_TUNE_GENERIC_Z | FFTB_TUNE_GENERIC_PLANE | FFTB_TUNE_FUSED | FFTB_TUNE_NO_L2_HINTS | FFTB_TUNE_HOST_DEFER)) return FFTB_EINVAL;
    if (tune && (tune->workspace_bytes < 0 || tune->ring_bands < 0 || tune->lead_bands < 0 || tune->z_ctas > 1024)) return FFTB_EINVAL;
    const bool dense = (desc->flags & FFTB_FLAG_DENSE) != 0;
    if (xm && (dense || xm->n < 1 || xm->n > (int64_t)1 << 24 || !xm->k1 || !xm->k2 || !xm->k3lo || !xm->len)) return FFTB_EINVAL;
    if (desc->flags & ~(uint32_t)(FFTB_FLAG_DENSE | FFTB_FLAG_BATCH_FASTEST)) return FFTB_EINVAL;
    const bool bf = (desc->flags & FFTB_FLAG_BATCH_FASTEST) != 0;
    if (bf && dense) return FFTB_EINVAL;
    if (desc->dtype != FFTB_C64 && desc->dtype != FFTB_C128) return FFTB_EINVAL;
    if (desc->scale != FFTB_SCALE_NONE && desc->scale != FFTB_SCALE_FORWARD) return FFTB_EINVAL;
    if (desc->batch < 1) return FFTB_EINVAL;
    for (int d = 0; d < 3; ++d) {
        if (desc->n[d] < 1) return FFTB_EINVAL;
        if (!dense && !xm && (desc->cutoff[d] < 0 || 2 * (long long)desc->cutoff[d] >= desc->n[d])) return FFTB_EINVAL;
    }
    if (xm) {
        // every point inside [-N_d/2, N_d/2) (EINVAL otherwise), strictly ascending (k1, k2), len >= 1
        for (int64_t s = 0; s < xm->n; ++s) {
            const long long lo = xm->k3lo[s], hi = lo + xm->len[s] - 1;
            if (xm->len[s] < 1) return FFTB_EINVAL;
            if (2 * (long long)xm->k1[s] < -desc->n[0] || 2 * (long long)xm->k1[s] >= desc->n[0]) return FFTB_EINVAL;
            if (2 * (long long)xm->k2[s] < -desc->n[1] || 2 * (long long)xm->k2[s] >= desc->n[1]) return FFTB_EINVAL;
            if (2 * lo < -desc->n[2] || 2 * hi >= desc->n[2]) return FFTB_EINVAL;
            if (s > 0 && !(xm->k1[s - 1] < xm->k1[s] || (xm->k1[s - 1] == xm->k1[s] && xm->k2[s - 1] < xm->k2[s]))) return FFTB_EINVAL;
        }
    }
    // predefined patterns.  A cut-off (or explicit map) that reaches beyond N_d/4 on some axis is no half-band problem any
    // more: such plans run on the full-band axis patterns of the dense plans (generic kernels, complex128), with their
    // pruned stick map.  N1 != N2: generic plane kernel, a few predefined pairs.
    bool wide = false;
    if (!dense && !xm)
        for (int d = 0; d < 3; ++d) wide = wide || 4 * (long long)desc->cutoff[d] > desc->n[d];
    if (xm)
        for (int64_t s = 0; s < xm->n; ++s) {
            const long long lo = xm->k3lo[s], hi = lo + xm->len[s] - 1;
            wide = wide || 4 * llabs((long long)xm->k1[s]) > desc->n[0] || 4 * llabs((long long)xm->k2[s]) > desc->n[1] || 4 * lo < -desc->n[2] ||
                   4 * hi > desc->n[2];
        }
    const bool full_band = dense || wide, rect = desc->n[0] != desc->n[1];
    if (bf && wide) return FFTB_EUNSUPPORTED;
    ZLaunch zl;
    PlaneLaunch plk;
    bool fast_plane = false;
    // dense cubes of 64, 128, 256 points: the line-pass kernel of fftb_dense.cuh (whole-batch launches)
    const bool dense_fast = dense && !(tflags & (FFTB_TUNE_GENERIC_Z | FFTB_TUNE_GENERIC_PLANE)) && find_dense_fast(desc->dtype, desc->n, &zl, &plk);
    if (dense_fast) fast_plane = true;
    else {
        if (!find_z(desc->dtype, desc->n[2], full_band, &zl)) return FFTB_EUNSUPPORTED;
        if (rect ? (full_band || !find_plane_xy(desc->dtype, desc->n[0], desc->n[1], &plk)) : !find_plane(desc->dtype, desc->n[0], full_band, &plk))
            return FFTB_EUNSUPPORTED;
    }
    const bool dense_cfg = full_band || rect; // no persistent kernels for these
    bool fast_z = false;
    {
        const bool gen_plane = (tflags & FFTB_TUNE_GENERIC_PLANE) != 0, gen_z = (tflags & FFTB_TUNE_GENERIC_Z) != 0;
        PlaneLaunch fast;
        if (!gen_plane && find_plane_fast(desc->dtype, desc->n[0], dense_cfg, &fast)) { plk = fast; fast_plane = true; }
        // 256 pattern: persistent plane kernels of their own (four-way split, fftb_plane_r4.cuh)
        if (!gen_plane && !dense_cfg && desc->n[0] == 256) {
            if (desc->dtype == FFTB_C128) {
                plk.run[MODE_INV] = &launch_plane_r4_inv<double>;
                plk.run[MODE_FWD] = &launch_plane_r4_fwd<double>;
                plk.run[MODE_VLOC] = &launch_plane_r4_vloc<double>;
            } else {
                plk.run[MODE_INV] = &launch_plane_r4_inv<float>;
                plk.run[MODE_FWD] = &launch_plane_r4_fwd<float>;
                plk.run[MODE_VLOC] = &launch_plane_r4_vloc<float>;
            }
            plk.ry = 1; // the forward and vloc kernels accumulate the four y residues into ONE plane of A themselves
            fast_plane = true; // persistent kernel: whole-batch launches (256 planes per band on 148 CTAs would waste half a wave)
        }
        ZLaunch zfast;
        if (!gen_z && find_z_fast(desc->dtype, desc->n[2], full_band, &zfast)) { zl = zfast; fast_z = true; }
    }
    // batch-fastest packed arrays: the transposition is folded into the persistent z passes, which must then exist
    if (bf && !(zl.batch_fastest && plk.ry == 1)) return FFTB_EUNSUPPORTED;
    FusedLaunch ful = {{0, 0, 0}, nullptr, nullptr};
    const bool fused = !bf && fast_plane && fast_z && (tflags & FFTB_TUNE_FUSED) && find_fused(desc->dtype, desc->n, dense, &ful);
    fftb_plan_s *p = new (std::nothrow) fftb_plan_s();
    if (!p) return FFTB_ENOMEM;
    try {
        p->desc = *desc;
        p->dense = dense;
        p->elem = desc->dtype == FFTB_C128 ? 16 : 8;
        p->zl = zl;
        p->plk = plk;
        p->ful = ful;
        p->fused = fused;
        p->bf = bf;
        p->l2_hints = (tflags & FFTB_TUNE_NO_L2_HINTS) ? 0 : 1;
        p->host_defer = (tflags & FFTB_TUNE_HOST_DEFER) != 0;
        p->z_ctas = tune ? (int)tune->z_ctas : 0;
        p->ry = plk.ry;
        const int n1 = desc->n[0], n2 = desc->n[1], n3 = desc->n[2];
        p->C = (int64_t)n1 * n2 * n3;
        int32_t a[3] = {desc->cutoff[0], desc->cutoff[1], desc->cutoff[2]};
        // ---- stick map: k1 major, k2 minor, both ascending over signed values (reading R5); either
        // generated from the cut-off (Eq. 9) or given explicitly
        std::vector<int32_t> ck1, ck2, clo, cln;
        p->nphantom = 0;
        if (xm) {
            // The kernels need (R6) one contiguous range of occupied k1 and one contiguous k2 run per k1.  A map with holes
            // gets them filled with zero-length PHANTOM sticks (a missing k1 column: one phantom at k2 = 0): no packed
            // point, a zero column of the intermediate in the inverse, a column nobody reads in the forward direction.
            for (int64_t s = 0; s < xm->n; ++s) {
                if (s > 0 && xm->k1[s] == xm->k1[s - 1])
                    for (int q2 = xm->k2[s - 1] + 1; q2 < xm->k2[s]; ++q2) { ck1.push_back(xm->k1[s]); ck2.push_back(q2); clo.push_back(0); cln.push_back(0); }
                else if (s > 0)
                    for (int q1 = xm->k1[s - 1] + 1; q1 < xm->k1[s]; ++q1) { ck1.push_back(q1); ck2.push_back(0); clo.push_back(0); cln.push_back(0); }
                ck1.push_back(xm->k1[s]); ck2.push_back(xm->k2[s]); clo.push_back(xm->k3lo[s]); cln.push_back(xm->len[s]);
            }
            p->nphantom = (int)((int64_t)ck1.size() - xm->n);
            a[0] = a[1] = a[2] = 0;
        } else {
            const int k1a = dense ? -(n1 / 2) : -a[0], k1b = dense ? (n1 + 1) / 2 - 1 : a[0];
            const int k2a = dense ? -(n2 / 2) : -a[1], k2b = dense ? (n2 + 1) / 2 - 1 : a[1];
            for (int q1 = k1a; q1 <= k1b; ++q1)
                for (int q2 = k2a; q2 <= k2b; ++q2) {
                    int lo, ln;
                    if (dense) {
                        lo = -(n3 / 2);
                        ln = n3;
                    } else {
                        if (!inside(q1, q2, 0, a)) continue;
                        int top = 0; // the column is symmetric in k3 and convex: grow from 0
                        while (top + 1 <= a[2] && inside(q1, q2, top + 1, a)) ++top;
                        lo = -top;
                        ln = 2 * top + 1;
                    }
                    ck1.push_back(q1); ck2.push_back(q2); clo.push_back(lo); cln.push_back(ln);
                }
        }
        if (ck1.empty()) { delete p; return FFTB_EUNSUPPORTED; }
        // the kernels need (R6): the occupied k1 form one contiguous range, the k2 of a k1 one contiguous run
        p->k1lo = ck1.front();
        p->nxocc = 0;
        int64_t run = 0;
        for (size_t s = 0; s < ck1.size();) {
            const int q1 = ck1[s];
            if (q1 != p->k1lo + p->nxocc) { delete p; return FFTB_EUNSUPPORTED; } // hole in the occupied k1 range
            const int first = (int)p->k1.size();
            int cnt = 0;
            for (; s < ck1.size() && ck1[s] == q1; ++s, ++cnt) {
                if (cnt > 0 && ck2[s] != ck2[s - 1] + 1) { delete p; return FFTB_EUNSUPPORTED; } // non-contiguous k2 run
                p->k1.push_back(q1);
                p->k2.push_back(ck2[s]);
                p->k3lo.push_back(clo[s]);
                p->len.push_back(cln[s]);
                p->off.push_back(run);
                run += cln[s];
            }
            int4 c;
            c.x = first; c.y = cnt; c.z = p->k2[first]; c.w = 0;
            p->h_col.push_back(c);
            ++p->nxocc;
        }
        p->off.push_back(run);
        p->S = run;
        p->nsticks = (int)p->k1.size();
        for (int c = 0; c < p->nxocc; ++c)
            if (p->h_col[c].y > 1) p->h_colperm.push_back(c);
        p->n_multi = (int)p->h_colperm.size();
        for (int c = 0; c < p->nxocc; ++c)
            if (p->h_col[c].y <= 1) p->h_colperm.push_back(c);
        if (p->S >= (int64_t)1 << 31) { delete p; return FFTB_EUNSUPPORTED; }
        memset(&p->tabs, 0, sizeof(p->tabs));
        if (p->nxocc <= FAST_MAXCOL)
            for (int c = 0; c < p->nxocc; ++c) { p->tabs.ct.col[c] = p->h_col[c]; p->tabs.ct.perm[c] = p->h_colperm[c]; }
        if (p->nxocc <= R4_MAXCOL)
            for (int c = 0; c < p->nxocc; ++c) { p->tabs.ct4.col[c] = p->h_col[c]; p->tabs.ct4.perm[c] = p->h_colperm[c]; }
        p->pitch = (int)align_up((size_t)p->nsticks, 16);
        p->h_stick.resize(p->nsticks);
        for (int s = 0; s < p->nsticks; ++s) {
            int4 v;
            v.x = (int)p->off[s]; v.y = p->k3lo[s]; v.z = p->len[s];
            v.w = (int)(((uint32_t)p->k1[s] & 0xffffu) | ((uint32_t)p->k2[s] << 16));
            p->h_stick[s] = v;
        }
        // ---- twiddle tables exp(+j 2 pi i / N), computed in long double, rounded once
        for (int d = 0; d < 3; ++d) {
            const int n = desc->n[d];
            p->h_tw[d].resize((size_t)n * p->elem);
            for (int i = 0; i < n; ++i) {
                // reduce to the first octant for accuracy
                const long double ang = 2.0L * 3.14159265358979323846264338327950288L * (long double)i / (long double)n;
                const long double c = cosl(ang), s = sinl(ang);
                if (p->elem == 16) {
                    double *t = reinterpret_cast<double *>(p->h_tw[d].data()) + 2 * (size_t)i;
                    t[0] = (double)c; t[1] = (double)s;
                } else {
                    float *t = reinterpret_cast<float *>(p->h_tw[d].data()) + 2 * (size_t)i;
                    t[0] = (float)c; t[1] = (float)s;
                }
            }
        }
        // ---- workspace: the plane-major intermediate for `chunk` bands.  The generic kernels are launched
        // per chunk and want it to stay in L2 between the two kernels of a chunk; the persistent fast
        // kernels gain more from few, long launches (measured on config 3: 48 MB -> 4.3 ms, whole batch
        // -> 3.9 ms per step), so their budget covers the whole batch whenever 4 GiB allow it.
        p->a_inv_stride = (long long)n3 * p->pitch;
        p->a_fwd_stride = (long long)p->ry * n3 * p->pitch;
        const size_t per_band = (size_t)(p->a_inv_stride + p->a_fwd_stride) * p->elem; // vloc needs both
        size_t budget = fast_plane ? (size_t)4 << 30 : (size_t)48 << 20;
        if (tune && tune->workspace_bytes > 0) budget = (size_t)tune->workspace_bytes;
        auto chunk_of = [&](size_t bytes_per_band) {
            long long c = (long long)(budget / bytes_per_band);
            if (c < 1) c = 1;
            if (c > desc->batch) c = desc->batch;
            return (int)c;
        };
        p->chunk = chunk_of(per_band);
        p->chunk_inv = chunk_of((size_t)p->a_inv_stride * p->elem);
        p->chunk_fwd = chunk_of((size_t)p->a_fwd_stride * p->elem);
        size_t o = 0;
        p->o_stick = o; o = align_up(o + sizeof(int4) * p->h_stick.size(), 256);
        p->o_col = o; o = align_up(o + sizeof(int4) * p->h_col.size(), 256);
        for (int d = 0; d < 3; ++d) { p->o_tw[d] = o; o = align_up(o + p->h_tw[d].size(), 256); }
        p->o_perm = o; o = align_up(o + sizeof(int) * p->h_colperm.size(), 256);
        p->o_sync = o; o = align_up(o + 2 * sizeof(int) * (size_t)desc->batch, 256); // per-band counters of the fused launches
        {
            size_t ws = (size_t)desc->batch * per_band;
            if (ws > budget) ws = budget;
            if (ws < per_band) ws = per_band;
            // fused launches: a ring of band slots at the start of the workspace that stays in L2 (4 x 6.7 MB at 128^3
            // complex128), producers 2 bands ahead of their consumers; nslot > lead >= 0 (fftb_fused.cuh)
            p->ring_ntiles = fused ? (p->nsticks + ful.geom.ts - 1) / ful.geom.ts : 0;
            p->ring_slot = fused ? (long long)p->ring_ntiles * ful.geom.tile : 0;
            const size_t slot = fused ? (size_t)p->ring_slot * p->elem : (size_t)p->a_inv_stride * p->elem;
            long long ring = tune && tune->ring_bands > 0 ? tune->ring_bands : 0, lead = tune && tune->lead_bands > 0 ? tune->lead_bands : 2;
            if (ring == 0) ring = lead + 2; // measured (profiles/r02_fused_ring_sweep.md): the smaller the ring, the less of it leaks to DRAM
            if (ring > desc->batch) ring = desc->batch;
            if (fused && ws < (size_t)ring * slot && (size_t)ring * slot <= budget) ws = (size_t)ring * slot; // tile-major slots are a little larger
            if (fused && ws < slot) ws = slot;
            if (ring > (long long)(ws / slot)) ring = (long long)(ws / slot);
            if (lead > ring - 1) lead = ring - 1;
            p->o_ws = o; o = align_up(o + ws, 256);
            p->ring_bands = (int)ring;
            p->lead_bands = (int)lead;
        }
        p->bytes_min = o;
        // two staging areas of the *_host calls: packed arrays arriving from the host and leaving for it (separate, so that
        // the next call's host-to-device copies run while this call's device-to-host copies are still under way)
        // (FFTB_TUNE_HOST_DEFER: two of each, taken in turn, so that the next call's transforms run while this call's results leave)
        const size_t area = (size_t)desc->batch * (size_t)p->S * p->elem;
        p->o_stage[0] = o; o = align_up(o + area, 256);
        p->o_stage_out[0] = o; o = align_up(o + area, 256);
        p->o_stage[1] = p->o_stage[0];
        p->o_stage_out[1] = p->o_stage_out[0];
        if (p->host_defer) {
            p->o_stage[1] = o; o = align_up(o + area, 256);
            p->o_stage_out[1] = o; o = align_up(o + area, 256);
        }
        p->bytes_stage = o;
        p->d_mem = nullptr;
        p->staging = false;
        p->pipe_ok = false;
        p->in_free_recorded[0] = p->in_free_recorded[1] = false;
        p->done_recorded[0] = p->done_recorded[1] = false;
        p->host_in_calls = p->host_out_calls = 0;
        p->sticky = 0;
        p->launches = 0;
        p->prof = false;
        p->ev_used = 0;
    } catch (const std::bad_alloc &) {
        delete p;
        return FFTB_ENOMEM;
    }
    *out = p;
    return FFTB_OK;
}

int fftb_plan_create(fftb_plan *out, const fftb_plan_desc *desc) { return plan_create_impl(out, desc, nullptr, nullptr); }

int fftb_plan_create_tuned(fftb_plan *out, const fftb_plan_desc *desc, const fftb_plan_tuning *tuning)
{
    return plan_create_impl(out, desc, nullptr, tuning);
}

int fftb_plan_create_explicit(fftb_plan *out, const fftb_plan_desc *desc, int64_t n_sticks, const int32_t *k1, const int32_t *k2,
                              const int32_t *k3lo, const int32_t *len)
{
    const ExplicitMap xm = {n_sticks, k1, k2, k3lo, len};
    return plan_create_impl(out, desc, &xm, nullptr);
}

int fftb_plan_create_explicit_tuned(fftb_plan *out, const fftb_plan_desc *desc, int64_t n_sticks, const int32_t *k1, const int32_t *k2,
                                    const int32_t *k3lo, const int32_t *len, const fftb_plan_tuning *tuning)
{
    const ExplicitMap xm = {n_sticks, k1, k2, k3lo, len};
    return plan_create_impl(out, desc, &xm, tuning);
}

int fftb_plan_info_get(fftb_plan p, fftb_plan_info *info)
{
    if (!p || !info) return FFTB_EINVAL;
    info->n_points = p->S;
    info->n_sticks = p->nsticks - p->nphantom;
    info->n_xocc = p->nxocc;
    info->device_bytes = (int64_t)p->bytes_min;
    info->device_bytes_host = (int64_t)p->bytes_stage;
    info->chunk_bands = p->chunk_inv;
    info->chunk_bands_fwd = p->chunk_fwd;
    info->chunk_bands_vloc = p->chunk;
    info->min_bytes_per_band_dir = (p->S + p->C) * (int64_t)p->elem;
    info->workspace_offset = (int64_t)p->o_ws;
    info->pitch = p->pitch;
    info->y_residues = p->ry;
    info->ring_bands = p->fused ? p->ring_bands : 0;
    info->lead_bands = p->fused ? p->lead_bands : 0;
    info->ring_tile_sticks = p->fused ? p->ful.geom.ts : 0;
    info->ring_tile_elems = p->fused ? p->ful.geom.tile : 0;
    info->ring_pair_pitch = p->fused ? p->ful.geom.rp : 0;
    return FFTB_OK;
}

int fftb_plan_get_map(fftb_plan p, int32_t *k1, int32_t *k2, int32_t *k3lo, int32_t *len, int64_t *off)
{
    if (!p) return FFTB_EINVAL;
    const size_t n = (size_t)p->nsticks;
    if (p->nphantom) { // the caller's map: the phantom sticks that fill its holes are left out
        size_t o = 0;
        for (size_t s = 0; s < n; ++s) {
            if (p->len[s] == 0) continue;
            if (k1) k1[o] = p->k1[s];
            if (k2) k2[o] = p->k2[s];
            if (k3lo) k3lo[o] = p->k3lo[s];
            if (len) len[o] = p->len[s];
            if (off) off[o] = p->off[s];
            ++o;
        }
        if (off) off[o] = p->off[n];
        return FFTB_OK;
    }
    if (k1) memcpy(k1, p->k1.data(), n * sizeof(int32_t));
    if (k2) memcpy(k2, p->k2.data(), n * sizeof(int32_t));
    if (k3lo) memcpy(k3lo, p->k3lo.data(), n * sizeof(int32_t));
    if (len) memcpy(len, p->len.data(), n * sizeof(int32_t));
    if (off) memcpy(off, p->off.data(), (n + 1) * sizeof(int64_t));
    return FFTB_OK;
}

int fftb_plan_bind(fftb_plan p, void *d_mem, size_t bytes, void *stream)
{
    if (!p || !d_mem) return FFTB_EINVAL;
    if ((uintptr_t)d_mem % 256) return FFTB_EINVAL;
    if (bytes < p->bytes_min) return FFTB_ENOMEM;
    if (p->sticky) return p->sticky;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned char *m = (unsigned char *)d_mem;
    cudaError_t e = cudaMemcpyAsync(m + p->o_stick, p->h_stick.data(), sizeof(int4) * p->h_stick.size(), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(m + p->o_col, p->h_col.data(), sizeof(int4) * p->h_col.size(), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(m + p->o_perm, p->h_colperm.data(), sizeof(int) * p->h_colperm.size(), cudaMemcpyHostToDevice, st);
    for (int d = 0; d < 3 && e == cudaSuccess; ++d)
        e = cudaMemcpyAsync(m + p->o_tw[d], p->h_tw[d].data(), p->h_tw[d].size(), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) { p->sticky = FFTB_ECUDA; return FFTB_ECUDA; }
    p->d_mem = m;
    p->staging = bytes >= p->bytes_stage;
    if (p->staging && !p->pipe_ok) {
        bool ok = cudaStreamCreateWithFlags(&p->cs_in, cudaStreamNonBlocking) == cudaSuccess &&
                  cudaStreamCreateWithFlags(&p->cs_out, cudaStreamNonBlocking) == cudaSuccess &&
                  cudaEventCreateWithFlags(&p->hev_in_free[0], cudaEventDisableTiming) == cudaSuccess &&
                  cudaEventCreateWithFlags(&p->hev_in_free[1], cudaEventDisableTiming) == cudaSuccess &&
                  cudaEventCreateWithFlags(&p->hev_done[0], cudaEventDisableTiming) == cudaSuccess &&
                  cudaEventCreateWithFlags(&p->hev_done[1], cudaEventDisableTiming) == cudaSuccess;
        for (int i = 0; i < 8 && ok; ++i)
            ok = cudaEventCreateWithFlags(&p->hev_in[i], cudaEventDisableTiming) == cudaSuccess &&
                 cudaEventCreateWithFlags(&p->hev_out[i], cudaEventDisableTiming) == cudaSuccess;
        if (!ok) { p->sticky = FFTB_ECUDA; return FFTB_ECUDA; }
        p->pipe_ok = true;
    }
    DevPlan &dv = p->dev;
    {
        int dev = 0, sms = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) {
            p->sticky = FFTB_ECUDA;
            return FFTB_ECUDA;
        }
        dv.sms = sms;
    }
    dv.n1 = p->desc.n[0]; dv.n2 = p->desc.n[1]; dv.n3 = p->desc.n[2];
    dv.nsticks = p->nsticks; dv.pitch = p->pitch; dv.nxocc = p->nxocc; dv.k1lo = p->k1lo; dv.ry = p->ry;
    dv.stick = (const int4 *)(m + p->o_stick);
    dv.col = (const int4 *)(m + p->o_col);
    dv.colperm = (const int *)(m + p->o_perm);
    dv.n_multi = p->n_multi;
    dv.tw1 = m + p->o_tw[0]; dv.tw2 = m + p->o_tw[1]; dv.tw3 = m + p->o_tw[2];
    dv.S = p->S;
    dv.scale = p->desc.scale == FFTB_SCALE_FORWARD ? 1.0 / (double)p->C : 1.0;
    if (p->fused) {
        // the ring as a tensor of 8-byte units: TS elements of a row | row parity | row pair | tile | slot (fftb_fused.cuh)
        const FusedGeom &ge = p->ful.geom;
        const cuuint64_t unit = p->elem / 8;
        const cuuint64_t dims[5] = {(cuuint64_t)ge.ts * unit, 2, (cuuint64_t)p->desc.n[2] / 2, (cuuint64_t)p->ring_ntiles, (cuuint64_t)p->ring_bands};
        const cuuint64_t strides[4] = {(cuuint64_t)ge.ts * p->elem, (cuuint64_t)ge.rp * p->elem, (cuuint64_t)ge.tile * p->elem,
                                       (cuuint64_t)p->ring_slot * p->elem};
        const cuuint32_t box[5] = {(cuuint32_t)(ge.ts * unit), 1, 1, (cuuint32_t)p->ring_ntiles, 1};
        const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
        typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                      const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                      CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
            qres != cudaDriverEntryPointSuccess || p->ring_ntiles > 256 ||
            ((encode_fn)fn)(&p->ring_map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 5, m + p->o_ws, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                            CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) {
            cudaGetLastError();
            p->fused = false; // the separate launches need nothing of the kind
        }
    }
    return FFTB_OK;
}

// packed arrays: 16-byte aligned; cuboids: 32-byte aligned for complex128 (the plane kernels move (x, x+1) pairs as
// one 32-byte access), 16-byte aligned for complex64
static int check_exec(fftb_plan p, const void *packed, const void *cuboid, int nb)
{
    if (!p || !packed || (!cuboid && nb >= 0)) return FFTB_EINVAL;
    if (p->sticky) return p->sticky;
    if (!p->d_mem) return FFTB_ESTATE;
    const int n = nb < 0 ? -nb : nb; // nb < 0: no cuboid operand (apply_vloc checks its second packed array itself)
    if (n < 1 || n > p->desc.batch) return FFTB_EINVAL;
    if ((uintptr_t)packed % 16) return FFTB_EINVAL;
    if (cuboid && (uintptr_t)cuboid % (p->elem == 16 ? 32 : 16)) return FFTB_EINVAL;
    return FFTB_OK;
}

int fftb_inverse(fftb_plan p, const void *d_packed, void *d_cuboid, int nb, void *stream)
{
    int rc = check_exec(p, d_packed, d_cuboid, nb);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned char *A = p->d_mem + p->o_ws;
    p->launches = 0;
    if (p->fused) { // one cooperative launch: z tiles and planes of the whole batch, A in a ring of band slots (L2)
        prof_begin(p, K_FUSED_INV, st);
        rc = p->ful.inv(p->dev, p->tabs, d_packed, A, p->ring_map, d_cuboid, p->ring_slot, nb, p->ring_bands, p->lead_bands, p->z_ctas, p->l2_hints,
                        (int *)(p->d_mem + p->o_sync), st);
        prof_end(p, st);
        if (rc) { p->sticky = rc; return rc; }
        p->launches = 1;
        return FFTB_OK;
    }
    for (int b0 = 0; b0 < nb; b0 += p->chunk_inv) {
        const int nc = nb - b0 < p->chunk_inv ? nb - b0 : p->chunk_inv;
        const unsigned char *pk = (const unsigned char *)d_packed + (p->bf ? (size_t)b0 : (size_t)b0 * p->S) * p->elem;
        unsigned char *cb = (unsigned char *)d_cuboid + (size_t)b0 * p->C * p->elem;
        prof_begin(p, K_ZINV, st);
        rc = p->zl.inv(p->dev, pk, A, p->a_inv_stride, nc, p->bf ? nb : 0, st);
        prof_end(p, st);
        prof_begin(p, K_PLANE_INV, st);
        if (!rc) rc = p->plk.run[MODE_INV](p->dev, p->tabs, A, nullptr, nullptr, cb, nullptr, p->a_inv_stride, 0, nc, st);
        prof_end(p, st);
        if (rc) { p->sticky = rc; return rc; }
        p->launches += 1 + p->plk.nkern[MODE_INV];
    }
    return FFTB_OK;
}

int fftb_forward(fftb_plan p, const void *d_cuboid, void *d_packed, int nb, void *stream)
{
    int rc = check_exec(p, d_packed, d_cuboid, nb);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned char *A = p->d_mem + p->o_ws;
    p->launches = 0;
    if (p->fused) {
        prof_begin(p, K_FUSED_FWD, st);
        rc = p->ful.fwd(p->dev, p->tabs, d_cuboid, A, d_packed, p->ring_slot, nb, p->ring_bands, p->lead_bands, p->z_ctas, p->l2_hints,
                        (int *)(p->d_mem + p->o_sync), st);
        prof_end(p, st);
        if (rc) { p->sticky = rc; return rc; }
        p->launches = 1;
        return FFTB_OK;
    }
    for (int b0 = 0; b0 < nb; b0 += p->chunk_fwd) {
        const int nc = nb - b0 < p->chunk_fwd ? nb - b0 : p->chunk_fwd;
        unsigned char *pk = (unsigned char *)d_packed + (p->bf ? (size_t)b0 : (size_t)b0 * p->S) * p->elem;
        const unsigned char *cb = (const unsigned char *)d_cuboid + (size_t)b0 * p->C * p->elem;
        prof_begin(p, K_PLANE_FWD, st);
        rc = p->plk.run[MODE_FWD](p->dev, p->tabs, nullptr, A, cb, nullptr, nullptr, 0, p->a_fwd_stride, nc, st);
        prof_end(p, st);
        prof_begin(p, K_ZFWD, st);
        if (!rc) rc = p->zl.fwd(p->dev, A, pk, p->a_fwd_stride, nc, p->bf ? nb : 0, st);
        prof_end(p, st);
        if (rc) { p->sticky = rc; return rc; }
        p->launches += 1 + p->plk.nkern[MODE_FWD];
    }
    return FFTB_OK;
}

int fftb_apply_vloc(fftb_plan p, const void *d_in, void *d_out, const void *d_vloc, int nb, void *stream)
{
    int rc = check_exec(p, d_in, nullptr, -nb);
    if (rc) return rc;
    if (!d_out || (uintptr_t)d_out % 16) return FFTB_EINVAL;
    if (!d_vloc || (uintptr_t)d_vloc % 16) return FFTB_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned char *Ai = p->d_mem + p->o_ws;
    unsigned char *Af = Ai + (size_t)p->chunk * p->a_inv_stride * p->elem;
    p->launches = 0;
    for (int b0 = 0; b0 < nb; b0 += p->chunk) {
        const int nc = nb - b0 < p->chunk ? nb - b0 : p->chunk;
        const unsigned char *pi = (const unsigned char *)d_in + (p->bf ? (size_t)b0 : (size_t)b0 * p->S) * p->elem;
        unsigned char *po = (unsigned char *)d_out + (p->bf ? (size_t)b0 : (size_t)b0 * p->S) * p->elem;
        prof_begin(p, K_ZINV, st);
        rc = p->zl.inv(p->dev, pi, Ai, p->a_inv_stride, nc, p->bf ? nb : 0, st);
        prof_end(p, st);
        prof_begin(p, K_PLANE_VLOC, st);
        if (!rc) rc = p->plk.run[MODE_VLOC](p->dev, p->tabs, Ai, Af, nullptr, nullptr, d_vloc, p->a_inv_stride, p->a_fwd_stride, nc, st);
        prof_end(p, st);
        prof_begin(p, K_ZFWD, st);
        if (!rc) rc = p->zl.fwd(p->dev, Af, po, p->a_fwd_stride, nc, p->bf ? nb : 0, st);
        prof_end(p, st);
        if (rc) { p->sticky = rc; return rc; }
        p->launches += 2 + p->plk.nkern[MODE_VLOC];
    }
    return FFTB_OK;
}

static int check_host(fftb_plan p, int nb)
{
    if (!p) return FFTB_EINVAL;
    if (p->sticky) return p->sticky;
    if (!p->d_mem) return FFTB_ESTATE;
    if (!p->staging) return FFTB_ENOMEM;
    if (nb < 1 || nb > p->desc.batch) return FFTB_EINVAL;
    return FFTB_OK;
}

// Band chunks of the *_host calls.
static int host_chunks(fftb_plan p, int nb)
{
    // at least 1024 z-planes per chunk keep the persistent kernels efficient; at most 4 chunks
    if (!p->pipe_ok || p->bf) return 1; // a band chunk of a batch-fastest array is no contiguous piece of host memory
    long long k = (long long)nb * p->desc.n[2] / 1024;
    if (k > 4) k = 4;
    if (k > nb) k = nb;
    if (p->elem == 8 && k > nb / 2) k = nb / 2; // chunks start on even bands (host_chunk_start)
    return k < 1 ? 1 : (int)k;
}
// first band of chunk k of K: with 8-byte elements and an odd S a chunk must start on an even band, so that the
// pointers handed to the device-pointer calls stay 16-byte aligned
static int host_chunk_start(fftb_plan p, int nb, int k, int K)
{
    if (k >= K) return nb;
    int b = (int)((long long)nb * k / K);
    if (p->elem == 8) b &= ~1;
    return b;
}
#define FFTB_CU(call) do { if ((call) != cudaSuccess) { p->sticky = FFTB_ECUDA; return FFTB_ECUDA; } } while (0)

// The incoming staging area may be refilled once the kernels of the call that read it last are done (not: once
// everything queued on the caller's stream is done -- that would put this call's host-to-device copies behind the
// previous call's device-to-host copies, and PCIe would never carry both directions at once).
// FFTB_TUNE_HOST_DEFER: successive calls take the two incoming (and the two outgoing) areas in turn.
static int host_in_area(fftb_plan p) { return p->host_defer ? (int)(p->host_in_calls++ & 1u) : 0; }
static int host_out_area(fftb_plan p) { return p->host_defer ? (int)(p->host_out_calls++ & 1u) : 0; }
static int host_in_begin(fftb_plan p, int a)
{
    if (p->in_free_recorded[a]) FFTB_CU(cudaStreamWaitEvent(p->cs_in, p->hev_in_free[a], 0));
    return FFTB_OK;
}
static int host_in_end(fftb_plan p, cudaStream_t st, int a)
{
    if (!p->pipe_ok) return FFTB_OK;
    FFTB_CU(cudaEventRecord(p->hev_in_free[a], st));
    p->in_free_recorded[a] = true;
    return FFTB_OK;
}
// An outgoing area may be rewritten once the device-to-host copies of the call that used it last are done.  Without
// FFTB_TUNE_HOST_DEFER that is implied (every call ends by making the caller's stream wait for its copies).
static int host_out_begin(fftb_plan p, cudaStream_t st, int a)
{
    if (p->host_defer && p->done_recorded[a]) FFTB_CU(cudaStreamWaitEvent(st, p->hev_done[a], 0));
    return FFTB_OK;
}
// The call completes, in the caller's stream order, when its last chunk is in host memory (which also keeps the outgoing
// area from being rewritten too early) -- unless completion is deferred to fftb_host_flush.
static int host_out_end(fftb_plan p, cudaStream_t st, cudaStream_t copies, int a)
{
    FFTB_CU(cudaEventRecord(p->hev_done[a], copies));
    p->done_recorded[a] = true;
    if (!p->host_defer) FFTB_CU(cudaStreamWaitEvent(st, p->hev_done[a], 0));
    return FFTB_OK;
}

int fftb_host_flush(fftb_plan p, void *stream)
{
    if (!p) return FFTB_EINVAL;
    if (p->sticky) return p->sticky;
    if (!p->d_mem) return FFTB_ESTATE;
    cudaStream_t st = (cudaStream_t)stream;
    for (int a = 0; a < 2; ++a)
        if (p->pipe_ok && p->done_recorded[a]) FFTB_CU(cudaStreamWaitEvent(st, p->hev_done[a], 0));
    return FFTB_OK;
}

int fftb_inverse_host(fftb_plan p, const void *h_packed, void *d_cuboid, int nb, void *stream)
{
    int rc = check_host(p, nb);
    if (rc) return rc;
    if (!h_packed || !d_cuboid) return FFTB_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const int ai = host_in_area(p);
    unsigned char *stg = p->d_mem + p->o_stage[ai];
    const int K = host_chunks(p, nb);
    const size_t band = (size_t)p->S * p->elem, cband = (size_t)p->C * p->elem;
    if (K == 1) {
        FFTB_CU(cudaMemcpyAsync(stg, h_packed, (size_t)nb * band, cudaMemcpyHostToDevice, st));
        rc = fftb_inverse(p, stg, d_cuboid, nb, stream);
        return rc ? rc : host_in_end(p, st, ai);
    }
    if ((rc = host_in_begin(p, ai))) return rc;
    int launches = 0;
    for (int k = 0; k < K; ++k) {
        const int b0 = host_chunk_start(p, nb, k, K), b1 = host_chunk_start(p, nb, k + 1, K);
        FFTB_CU(cudaMemcpyAsync(stg + b0 * band, (const unsigned char *)h_packed + b0 * band, (size_t)(b1 - b0) * band,
                                cudaMemcpyHostToDevice, p->cs_in));
        FFTB_CU(cudaEventRecord(p->hev_in[k], p->cs_in));
        FFTB_CU(cudaStreamWaitEvent(st, p->hev_in[k], 0));
        rc = fftb_inverse(p, stg + b0 * band, (unsigned char *)d_cuboid + b0 * cband, b1 - b0, stream);
        if (rc) return rc;
        launches += p->launches;
    }
    p->launches = launches;
    return host_in_end(p, st, ai);
}

int fftb_forward_host(fftb_plan p, const void *d_cuboid, void *h_packed, int nb, void *stream)
{
    int rc = check_host(p, nb);
    if (rc) return rc;
    if (!h_packed || !d_cuboid) return FFTB_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const int ao = host_out_area(p);
    unsigned char *stg = p->d_mem + p->o_stage_out[ao];
    const int K = host_chunks(p, nb);
    const size_t band = (size_t)p->S * p->elem, cband = (size_t)p->C * p->elem;
    if ((rc = host_out_begin(p, st, ao))) return rc;
    if (K == 1) {
        rc = fftb_forward(p, d_cuboid, stg, nb, stream);
        if (rc) return rc;
        if (!p->host_defer || !p->pipe_ok) {
            FFTB_CU(cudaMemcpyAsync(h_packed, stg, (size_t)nb * band, cudaMemcpyDeviceToHost, st));
            return FFTB_OK;
        }
        // deferred completion: the copy leaves on the plan's own stream
        FFTB_CU(cudaEventRecord(p->hev_out[0], st));
        FFTB_CU(cudaStreamWaitEvent(p->cs_out, p->hev_out[0], 0));
        FFTB_CU(cudaMemcpyAsync(h_packed, stg, (size_t)nb * band, cudaMemcpyDeviceToHost, p->cs_out));
        return host_out_end(p, st, p->cs_out, ao);
    }
    int launches = 0;
    for (int k = 0; k < K; ++k) {
        const int b0 = host_chunk_start(p, nb, k, K), b1 = host_chunk_start(p, nb, k + 1, K);
        rc = fftb_forward(p, (const unsigned char *)d_cuboid + b0 * cband, stg + b0 * band, b1 - b0, stream);
        if (rc) return rc;
        launches += p->launches;
        FFTB_CU(cudaEventRecord(p->hev_out[k], st));
        FFTB_CU(cudaStreamWaitEvent(p->cs_out, p->hev_out[k], 0));
        FFTB_CU(cudaMemcpyAsync((unsigned char *)h_packed + b0 * band, stg + b0 * band, (size_t)(b1 - b0) * band,
                                cudaMemcpyDeviceToHost, p->cs_out));
    }
    p->launches = launches;
    return host_out_end(p, st, p->cs_out, ao);
}

int fftb_apply_vloc_host(fftb_plan p, const void *h_in, void *h_out, const void *d_vloc, int nb, void *stream)
{
    int rc = check_host(p, nb);
    if (rc) return rc;
    if (!h_in || !h_out) return FFTB_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const int ai = host_in_area(p), ao = host_out_area(p);
    unsigned char *stg = p->d_mem + p->o_stage[ai], *sto = p->d_mem + p->o_stage_out[ao];
    const int K = host_chunks(p, nb);
    const size_t band = (size_t)p->S * p->elem;
    if ((rc = host_out_begin(p, st, ao))) return rc;
    if (K == 1) {
        FFTB_CU(cudaMemcpyAsync(stg, h_in, (size_t)nb * band, cudaMemcpyHostToDevice, st));
        rc = fftb_apply_vloc(p, stg, sto, d_vloc, nb, stream);
        if (rc) return rc;
        if (!p->host_defer || !p->pipe_ok) {
            FFTB_CU(cudaMemcpyAsync(h_out, sto, (size_t)nb * band, cudaMemcpyDeviceToHost, st));
            return host_in_end(p, st, ai);
        }
        if ((rc = host_in_end(p, st, ai))) return rc;
        FFTB_CU(cudaEventRecord(p->hev_out[0], st));
        FFTB_CU(cudaStreamWaitEvent(p->cs_out, p->hev_out[0], 0));
        FFTB_CU(cudaMemcpyAsync(h_out, sto, (size_t)nb * band, cudaMemcpyDeviceToHost, p->cs_out));
        return host_out_end(p, st, p->cs_out, ao);
    }
    if ((rc = host_in_begin(p, ai))) return rc;
    int launches = 0;
    for (int k = 0; k < K; ++k) {
        const int b0 = host_chunk_start(p, nb, k, K), b1 = host_chunk_start(p, nb, k + 1, K);
        FFTB_CU(cudaMemcpyAsync(stg + b0 * band, (const unsigned char *)h_in + b0 * band, (size_t)(b1 - b0) * band,
                                cudaMemcpyHostToDevice, p->cs_in));
        FFTB_CU(cudaEventRecord(p->hev_in[k], p->cs_in));
        FFTB_CU(cudaStreamWaitEvent(st, p->hev_in[k], 0));
        rc = fftb_apply_vloc(p, stg + b0 * band, sto + b0 * band, d_vloc, b1 - b0, stream);
        if (rc) return rc;
        launches += p->launches;
        FFTB_CU(cudaEventRecord(p->hev_out[k], st));
        FFTB_CU(cudaStreamWaitEvent(p->cs_out, p->hev_out[k], 0));
        FFTB_CU(cudaMemcpyAsync((unsigned char *)h_out + b0 * band, sto + b0 * band, (size_t)(b1 - b0) * band,
                                cudaMemcpyDeviceToHost, p->cs_out));
    }
    if ((rc = host_in_end(p, st, ai))) return rc;
    p->launches = launches;
    return host_out_end(p, st, p->cs_out, ao);
}

static int dense_move(fftb_plan pruned, fftb_plan dense, const void *src, void *dst, int nb, void *stream, bool extract)
{
    if (!pruned || !dense || !src || !dst) return FFTB_EINVAL;
    if (pruned->sticky) return pruned->sticky;
    if (!pruned->d_mem || !dense->dense || pruned->dense) return FFTB_ESTATE;
    for (int d = 0; d < 3; ++d)
        if (pruned->desc.n[d] != dense->desc.n[d]) return FFTB_ESTATE;
    if (pruned->desc.dtype != dense->desc.dtype) return FFTB_ESTATE;
    if (nb < 1 || nb > pruned->desc.batch || nb > dense->desc.batch) return FFTB_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    if (!extract && cudaMemsetAsync(dst, 0, (size_t)nb * dense->S * dense->elem, st) != cudaSuccess) return FFTB_ECUDA;
    dim3 grid((pruned->nsticks + 7) / 8, nb);
    const DevPlan &dv = pruned->dev;
    if (pruned->elem == 16)
        dense_embed_k<double><<<grid, 256, 0, st>>>(dv.stick, dv.nsticks, dv.S, (const double2 *)src, (double2 *)dst, dv.n1, dv.n2, dv.n3, extract);
    else
        dense_embed_k<float><<<grid, 256, 0, st>>>(dv.stick, dv.nsticks, dv.S, (const float2 *)src, (float2 *)dst, dv.n1, dv.n2, dv.n3, extract);
    pruned->launches = 1;
    return cudaGetLastError() == cudaSuccess ? FFTB_OK : FFTB_ECUDA;
}

int fftb_dense_embed(fftb_plan pruned, fftb_plan dense, const void *d_packed_pruned, void *d_packed_dense, int nb, void *stream)
{
    return dense_move(pruned, dense, d_packed_pruned, d_packed_dense, nb, stream, false);
}
int fftb_dense_extract(fftb_plan pruned, fftb_plan dense, const void *d_packed_dense, void *d_packed_pruned, int nb, void *stream)
{
    return dense_move(pruned, dense, d_packed_dense, d_packed_pruned, nb, stream, true);
}

int fftb_packed_transpose(fftb_plan p, const void *d_in, void *d_out, int nb, int to_band_slowest, void *stream)
{
    if (!p || !d_in || !d_out || d_in == d_out) return FFTB_EINVAL;
    if (p->sticky) return p->sticky;
    if (nb < 1 || (uintptr_t)d_in % 16 || (uintptr_t)d_out % 16) return FFTB_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    // to_band_slowest: in = [S][nb] -> out = [nb][S]; otherwise in = [nb][S] -> out = [S][nb]
    const long long R = to_band_slowest ? p->S : nb, Cn = to_band_slowest ? nb : p->S;
    const long long tiles = ((Cn + 31) / 32) * ((R + 31) / 32);
    if (tiles > 0x7fffffffLL) return FFTB_EUNSUPPORTED;
    const unsigned grid = (unsigned)tiles;
    if (p->elem == 16)
        transpose_k<double2><<<grid, 256, 0, st>>>((const double2 *)d_in, (double2 *)d_out, R, Cn);
    else
        transpose_k<float2><<<grid, 256, 0, st>>>((const float2 *)d_in, (float2 *)d_out, R, Cn);
    p->launches = 1;
    return cudaGetLastError() == cudaSuccess ? FFTB_OK : FFTB_ECUDA;
}

int fftb_plan_last_launches(fftb_plan p) { return p ? p->launches : FFTB_EINVAL; }

int fftb_probe_store_port(int n_sms, double *bytes_per_clk_per_sm, double *gbs)
{
    if (!bytes_per_clk_per_sm || n_sms < 1 || n_sms > 1024) return FFTB_EINVAL;
    const double v = probe_store_port(n_sms, gbs);
    if (v < 0.0) return FFTB_ECUDA;
    *bytes_per_clk_per_sm = v;
    return FFTB_OK;
}

int fftb_probe_fma(int dtype, double *tflops, double *ms)
{
    if (!tflops || (dtype != FFTB_C64 && dtype != FFTB_C128)) return FFTB_EINVAL;
    const double v = dtype == FFTB_C128 ? probe_fma_tflops<double>(ms) : probe_fma_tflops<float>(ms);
    if (v < 0.0) return FFTB_ECUDA;
    *tflops = v;
    return FFTB_OK;
}


int fftb_plan_profile(fftb_plan p, int enable)
{
    if (!p) return FFTB_EINVAL;
    p->prof = enable != 0;
    p->ev_used = 0;
    return FFTB_OK;
}

int fftb_plan_profile_read(fftb_plan p, double *ms, int64_t *count)
{
    if (!p || !ms || !count) return FFTB_EINVAL;
    for (int k = 0; k < K_KINDS; ++k) { ms[k] = 0.0; count[k] = 0; }
    for (size_t i = 0; i + 1 < p->ev_used; i += 2) {
        if (cudaEventSynchronize(p->ev[i + 1]) != cudaSuccess) return FFTB_ECUDA;
        float t = 0.f;
        if (cudaEventElapsedTime(&t, p->ev[i], p->ev[i + 1]) != cudaSuccess) return FFTB_ECUDA;
        ms[p->ev_kind[i / 2]] += t;
        count[p->ev_kind[i / 2]] += 1;
    }
    p->ev_used = 0;
    return FFTB_OK;
}

int fftb_plan_destroy(fftb_plan p)
{
    if (!p) return FFTB_EINVAL;
    for (cudaEvent_t e : p->ev) cudaEventDestroy(e);
    if (p->pipe_ok) {
        cudaStreamDestroy(p->cs_in);
        cudaStreamDestroy(p->cs_out);
        for (int i = 0; i < 2; ++i) { cudaEventDestroy(p->hev_in_free[i]); cudaEventDestroy(p->hev_done[i]); }
        for (int i = 0; i < 8; ++i) { cudaEventDestroy(p->hev_in[i]); cudaEventDestroy(p->hev_out[i]); }
    }
    delete p;
    return FFTB_OK;
}

// ------------------------------------------------------------------------------------------------
// fftb_inverse_static (include/fftb.h): the inverse transform for callers that may not allocate device memory.  The
// scratch the two kernels of a band chunk share -- the plane-major intermediate A -- and the plan's tables live in a
// file-scope device array instead of a caller-owned bind block.
//
// In HOST code the name g_static_scratch is only a stand-in for the symbol: it is not a device address, and a kernel
// handed `g_static_scratch` itself would fault (or, where the GPU can reach host memory, silently use the wrong memory).
// Its device address is looked up once per device with cudaGetSymbolAddress (that device current), kept in a small
// table under a mutex, and THAT pointer goes to the kernels.
// ------------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char g_static_scratch[FFTB_STATIC_SCRATCH_BYTES];

struct StaticScratch { unsigned char *ptr; int sms; };
static std::mutex g_static_mu;
static std::map<int, StaticScratch> g_static_dev; // device ordinal -> device address of g_static_scratch, SM count

static int static_scratch_current_device(StaticScratch *out)
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return FFTB_ECUDA; }
    std::lock_guard<std::mutex> lock(g_static_mu);
    auto it = g_static_dev.find(dev);
    if (it == g_static_dev.end()) {
        StaticScratch s = {nullptr, 0};
        if (cudaGetSymbolAddress((void **)&s.ptr, g_static_scratch) != cudaSuccess || !s.ptr || (uintptr_t)s.ptr % 256) {
            cudaGetLastError();
            return FFTB_ECUDA;
        }
        if (cudaDeviceGetAttribute(&s.sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || s.sms < 1) {
            cudaGetLastError();
            return FFTB_ECUDA;
        }
        it = g_static_dev.emplace(dev, s).first;
    }
    *out = it->second;
    return 0;
}

int fftb_inverse_static(fftb_plan p, const void *d_packed, void *d_cuboid, int nb, void *stream)
{
    if (!p || !d_packed || !d_cuboid) return FFTB_EINVAL;
    if (nb < 1 || nb > p->desc.batch) return FFTB_EINVAL;
    if ((uintptr_t)d_packed % 16 || (uintptr_t)d_cuboid % (p->elem == 16 ? 32 : 16)) return FFTB_EINVAL;
    // layout inside the array: the tables at the offsets they have in a bind block (all before o_sync), then A
    const size_t o_a = p->o_sync, band = (size_t)p->a_inv_stride * p->elem;
    if (o_a + band > (size_t)FFTB_STATIC_SCRATCH_BYTES) return FFTB_ETOOBIG;
    StaticScratch sc;
    if (int rc = static_scratch_current_device(&sc)) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned char *m = sc.ptr;
    // the array keeps whatever the last call (of any plan) left: rewrite the tables, every time.  A needs no clearing: the
    // z pass of a chunk writes every (z, stick) element the plane kernel of that chunk reads.
    cudaError_t e = cudaMemcpyAsync(m + p->o_stick, p->h_stick.data(), sizeof(int4) * p->h_stick.size(), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(m + p->o_col, p->h_col.data(), sizeof(int4) * p->h_col.size(), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(m + p->o_perm, p->h_colperm.data(), sizeof(int) * p->h_colperm.size(), cudaMemcpyHostToDevice, st);
    for (int d = 0; d < 3 && e == cudaSuccess; ++d)
        e = cudaMemcpyAsync(m + p->o_tw[d], p->h_tw[d].data(), p->h_tw[d].size(), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) { cudaGetLastError(); return FFTB_ECUDA; }
    DevPlan dv;
    dv.n1 = p->desc.n[0]; dv.n2 = p->desc.n[1]; dv.n3 = p->desc.n[2];
    dv.nsticks = p->nsticks; dv.pitch = p->pitch; dv.nxocc = p->nxocc; dv.k1lo = p->k1lo; dv.ry = p->ry;
    dv.stick = (const int4 *)(m + p->o_stick);
    dv.col = (const int4 *)(m + p->o_col);
    dv.colperm = (const int *)(m + p->o_perm);
    dv.n_multi = p->n_multi;
    dv.tw1 = m + p->o_tw[0]; dv.tw2 = m + p->o_tw[1]; dv.tw3 = m + p->o_tw[2];
    dv.S = p->S;
    dv.scale = p->desc.scale == FFTB_SCALE_FORWARD ? 1.0 / (double)p->C : 1.0;
    dv.sms = sc.sms;
    unsigned char *A = m + o_a;
    long long chunk = (long long)(((size_t)FFTB_STATIC_SCRATCH_BYTES - o_a) / band);
    if (chunk > nb) chunk = nb;
    for (int b0 = 0; b0 < nb; b0 += (int)chunk) {
        const int nc = nb - b0 < (int)chunk ? nb - b0 : (int)chunk;
        const unsigned char *pk = (const unsigned char *)d_packed + (p->bf ? (size_t)b0 : (size_t)b0 * p->S) * p->elem;
        unsigned char *cb = (unsigned char *)d_cuboid + (size_t)b0 * p->C * p->elem;
        int rc = p->zl.inv(dv, pk, A, p->a_inv_stride, nc, p->bf ? nb : 0, st);
        if (!rc) rc = p->plk.run[MODE_INV](dv, p->tabs, A, nullptr, nullptr, cb, nullptr, p->a_inv_stride, 0, nc, st);
        if (rc) return rc;
    }
    return FFTB_OK;
}

// ------------------------------------------------------------------------------------------------
// slab-distributed transform (include/fftb.h; fftb_slab.cuh): two ordinary plans -- the z passes on the own sticks
// (an explicit stick map, the whole z axis) and the plane passes on all sticks (run on the own z slab only) -- and
// the row-copy kernel between them
// ------------------------------------------------------------------------------------------------
struct fftb_slab_plan_s {
    int world, rank, batch, n3;
    size_t elem;
    fftb_plan zp, pp;
    std::vector<int64_t> stick_lo, packed_lo, z_lo; // world + 1 entries each
    size_t o_z, o_p, bytes;
    bool bound;
};

static int slab_pitch(int64_t nsticks) { return (int)((nsticks + 15) / 16 * 16); }

static int slab_copy(fftb_slab_plan p, const SlabSegs &sg, const void *src, int max_rows, int nb, cudaStream_t st)
{
    int rb = max_rows < 64 ? max_rows : 64;
    if (rb < 1) rb = 1;
    dim3 grid(rb, nb, sg.n);
    if (p->elem == 16) slab_rows_k<double2><<<grid, 256, 0, st>>>(sg, (const double2 *)src);
    else slab_rows_k<float2><<<grid, 256, 0, st>>>(sg, (const float2 *)src);
    return cudaGetLastError() == cudaSuccess ? FFTB_OK : FFTB_ECUDA;
}

int fftb_slab_plan_create(fftb_slab_plan *out, const fftb_plan_desc *desc, int world, int rank)
{
    if (!out || !desc) return FFTB_EINVAL;
    *out = nullptr;
    if (world < 1 || rank < 0 || rank >= world) return FFTB_EINVAL;
    if (world > SLAB_MAXR || desc->flags) return FFTB_EUNSUPPORTED;
    fftb_plan pp = nullptr;
    int rc = plan_create_impl(&pp, desc, nullptr, nullptr);
    if (rc) return rc;
    fftb_slab_plan_s *p = new (std::nothrow) fftb_slab_plan_s();
    if (!p) { fftb_plan_destroy(pp); return FFTB_ENOMEM; }
    p->world = world; p->rank = rank; p->batch = desc->batch; p->n3 = desc->n[2]; p->elem = pp->elem;
    p->pp = pp; p->zp = nullptr; p->bound = false;
    if (pp->nxocc < world || desc->n[2] < world || pp->ry != 1) { fftb_slab_plan_destroy(p); return FFTB_EUNSUPPORTED; }
    // sticks: contiguous ranges of occupied k1 columns, cut where the running stick count passes r * n_sticks / world
    p->stick_lo.assign(world + 1, 0);
    {
        int col = 0;
        for (int r = 1; r < world; ++r) {
            const int64_t target = (int64_t)r * pp->nsticks / world;
            int c = col + 1; // at least one column per rank
            while (c < pp->nxocc - (world - r) && pp->h_col[c].x < target) ++c;
            col = c;
            p->stick_lo[r] = pp->h_col[c].x;
        }
        p->stick_lo[world] = pp->nsticks;
    }
    p->packed_lo.resize(world + 1);
    p->z_lo.resize(world + 1);
    for (int r = 0; r <= world; ++r) {
        p->packed_lo[r] = pp->off[(size_t)p->stick_lo[r]];
        p->z_lo[r] = (int64_t)r * desc->n[2] / world;
    }
    // the own sticks as an explicit map (the whole z axis, the band count of the description)
    const int64_t s0 = p->stick_lo[rank], s1 = p->stick_lo[rank + 1];
    const ExplicitMap xm = {s1 - s0, pp->k1.data() + s0, pp->k2.data() + s0, pp->k3lo.data() + s0, pp->len.data() + s0};
    fftb_plan_desc dz = *desc;
    for (int d = 0; d < 3; ++d) dz.cutoff[d] = 0;
    rc = plan_create_impl(&p->zp, &dz, &xm, nullptr);
    if (!rc && (p->zp->ry != 1 || p->zp->chunk_inv < desc->batch || p->zp->chunk_fwd < desc->batch || pp->chunk_inv < desc->batch ||
                pp->chunk_fwd < desc->batch))
        rc = FFTB_EUNSUPPORTED; // the whole batch goes through the intermediates in one piece
    if (rc) { fftb_slab_plan_destroy(p); return rc; }
    p->o_z = 0;
    p->o_p = align_up(p->zp->bytes_min, 256);
    p->bytes = p->o_p + align_up(pp->bytes_min, 256);
    *out = p;
    return FFTB_OK;
}

int fftb_slab_plan_info_get(fftb_slab_plan p, fftb_slab_info *info)
{
    if (!p || !info) return FFTB_EINVAL;
    info->n_points_local = p->packed_lo[p->rank + 1] - p->packed_lo[p->rank];
    info->n_sticks_local = p->stick_lo[p->rank + 1] - p->stick_lo[p->rank];
    info->planes_local = p->z_lo[p->rank + 1] - p->z_lo[p->rank];
    info->device_bytes = (int64_t)p->bytes;
    info->n_points = p->pp->S;
    info->n_sticks = p->pp->nsticks;
    return FFTB_OK;
}

int fftb_slab_plan_counts(fftb_slab_plan p, int64_t *stick_lo, int64_t *packed_lo, int64_t *z_lo)
{
    if (!p) return FFTB_EINVAL;
    const size_t n = (size_t)p->world + 1;
    if (stick_lo) memcpy(stick_lo, p->stick_lo.data(), n * sizeof(int64_t));
    if (packed_lo) memcpy(packed_lo, p->packed_lo.data(), n * sizeof(int64_t));
    if (z_lo) memcpy(z_lo, p->z_lo.data(), n * sizeof(int64_t));
    return FFTB_OK;
}

int fftb_slab_plan_bind(fftb_slab_plan p, void *d_mem, size_t bytes, void *stream)
{
    if (!p || !d_mem) return FFTB_EINVAL;
    if ((uintptr_t)d_mem % 256) return FFTB_EINVAL;
    if (bytes < p->bytes) return FFTB_ENOMEM;
    unsigned char *m = (unsigned char *)d_mem;
    int rc = fftb_plan_bind(p->zp, m + p->o_z, p->o_p - p->o_z, stream);
    if (!rc) rc = fftb_plan_bind(p->pp, m + p->o_p, p->bytes - p->o_p, stream);
    p->bound = rc == FFTB_OK;
    return rc;
}

int fftb_slab_plan_exchange_ptr(fftb_slab_plan p, int which, void **d_ptr)
{
    if (!p || !d_ptr || (which != 0 && which != 1)) return FFTB_EINVAL;
    if (!p->bound) return FFTB_ESTATE;
    *d_ptr = which == 0 ? (void *)(p->pp->d_mem + p->pp->o_ws) : (void *)(p->zp->d_mem + p->zp->o_ws);
    return FFTB_OK;
}

static int slab_check(fftb_slab_plan p, const void *a, const void *b, bool need_b, int nb)
{
    if (!p || !a || (need_b && !b)) return FFTB_EINVAL;
    if (!p->bound) return FFTB_ESTATE;
    if (p->zp->sticky) return p->zp->sticky;
    if (p->pp->sticky) return p->pp->sticky;
    if (nb < 1 || nb > p->batch) return FFTB_EINVAL;
    if ((uintptr_t)a % 16 || (need_b && (uintptr_t)b % 16)) return FFTB_EINVAL;
    return FFTB_OK;
}

// segments of an exchange.  to_planes: rows = z-planes of the slab owner, columns = sticks of the stick owner (inverse);
// otherwise the forward direction.  send: this rank is the source of the rows (pack side), else the unpack side.
int fftb_slab_inverse_begin(fftb_slab_plan p, const void *d_packed_local, void *const *d_peer, void *d_send, int nb, void *stream)
{
    int rc = slab_check(p, d_packed_local, d_send, d_peer == nullptr, nb);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    fftb_plan zp = p->zp;
    unsigned char *A = zp->d_mem + zp->o_ws;
    rc = zp->zl.inv(zp->dev, d_packed_local, A, zp->a_inv_stride, nb, 0, st);
    if (rc) { zp->sticky = rc; return rc; }
    const int r = p->rank, R = p->world;
    const long long n_r = p->stick_lo[r + 1] - p->stick_lo[r], pitch_r = zp->pitch, pitch = p->pp->pitch;
    SlabSegs sg;
    sg.n = R;
    long long off = 0;
    int max_rows = 1;
    for (int d = 0; d < R; ++d) {
        const long long slab_d = p->z_lo[d + 1] - p->z_lo[d];
        SlabSeg &g = sg.s[d];
        g.rows = (int)slab_d; g.cols = (int)n_r; g.peer = d;
        g.src_off = p->z_lo[d] * pitch_r; g.src_sb = (long long)p->n3 * pitch_r; g.src_sr = pitch_r;
        if (d_peer) { // straight into peer d's intermediate A[band][own plane][all sticks]
            if (!d_peer[d]) return FFTB_EINVAL;
            sg.dst[d] = d_peer[d];
            g.dst_off = p->stick_lo[r]; g.dst_sb = slab_d * pitch; g.dst_sr = pitch;
        } else {      // staging buffer [peer][band][row][column]
            sg.dst[d] = d_send;
            g.dst_off = off; g.dst_sb = slab_d * n_r; g.dst_sr = n_r;
            off += (long long)nb * slab_d * n_r;
        }
        if (g.rows > max_rows) max_rows = g.rows;
    }
    return slab_copy(p, sg, A, max_rows, nb, st);
}

int fftb_slab_inverse_end(fftb_slab_plan p, const void *d_recv, void *d_cuboid_slab, int nb, void *stream)
{
    int rc = slab_check(p, d_cuboid_slab, nullptr, false, nb);
    if (rc) return rc;
    if ((uintptr_t)d_cuboid_slab % (p->elem == 16 ? 32 : 16) || (d_recv && (uintptr_t)d_recv % 16)) return FFTB_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    fftb_plan pp = p->pp;
    unsigned char *A = pp->d_mem + pp->o_ws;
    const int r = p->rank, R = p->world;
    const long long slab_r = p->z_lo[r + 1] - p->z_lo[r], pitch = pp->pitch;
    if (d_recv) { // [peer][band][own plane][the peer's sticks] -> A[band][own plane][all sticks]
        SlabSegs sg;
        sg.n = R;
        long long off = 0;
        for (int s = 0; s < R; ++s) {
            const long long n_s = p->stick_lo[s + 1] - p->stick_lo[s];
            SlabSeg &g = sg.s[s];
            g.rows = (int)slab_r; g.cols = (int)n_s; g.peer = s;
            g.src_off = off; g.src_sb = slab_r * n_s; g.src_sr = n_s;
            sg.dst[s] = A;
            g.dst_off = p->stick_lo[s]; g.dst_sb = slab_r * pitch; g.dst_sr = pitch;
            off += (long long)nb * slab_r * n_s;
        }
        rc = slab_copy(p, sg, d_recv, (int)slab_r, nb, st);
        if (rc) return rc;
    }
    DevPlan dv = pp->dev;
    dv.n3 = (int)slab_r; // the plane kernels walk the planes of the slab only
    rc = pp->plk.run[MODE_INV](dv, pp->tabs, A, nullptr, nullptr, d_cuboid_slab, nullptr, slab_r * pitch, 0, nb, st);
    if (rc) pp->sticky = rc;
    return rc;
}

int fftb_slab_forward_begin(fftb_slab_plan p, const void *d_cuboid_slab, void *const *d_peer, void *d_send, int nb, void *stream)
{
    int rc = slab_check(p, d_cuboid_slab, d_send, d_peer == nullptr, nb);
    if (rc) return rc;
    if ((uintptr_t)d_cuboid_slab % (p->elem == 16 ? 32 : 16)) return FFTB_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    fftb_plan pp = p->pp;
    unsigned char *A = pp->d_mem + pp->o_ws;
    const int r = p->rank, R = p->world;
    const long long slab_r = p->z_lo[r + 1] - p->z_lo[r], pitch = pp->pitch;
    DevPlan dv = pp->dev;
    dv.n3 = (int)slab_r;
    rc = pp->plk.run[MODE_FWD](dv, pp->tabs, nullptr, A, d_cuboid_slab, nullptr, nullptr, 0, slab_r * pitch, nb, st);
    if (rc) { pp->sticky = rc; return rc; }
    SlabSegs sg;
    sg.n = R;
    long long off = 0;
    for (int d = 0; d < R; ++d) {
        const long long n_d = p->stick_lo[d + 1] - p->stick_lo[d], pitch_d = slab_pitch(n_d);
        SlabSeg &g = sg.s[d];
        g.rows = (int)slab_r; g.cols = (int)n_d; g.peer = d;
        g.src_off = p->stick_lo[d]; g.src_sb = slab_r * pitch; g.src_sr = pitch;
        if (d_peer) { // straight into peer d's intermediate A[band][all planes][own sticks]
            if (!d_peer[d]) return FFTB_EINVAL;
            sg.dst[d] = d_peer[d];
            g.dst_off = p->z_lo[r] * pitch_d; g.dst_sb = (long long)p->n3 * pitch_d; g.dst_sr = pitch_d;
        } else {
            sg.dst[d] = d_send;
            g.dst_off = off; g.dst_sb = slab_r * n_d; g.dst_sr = n_d;
            off += (long long)nb * slab_r * n_d;
        }
    }
    return slab_copy(p, sg, A, (int)slab_r, nb, st);
}

int fftb_slab_forward_end(fftb_slab_plan p, const void *d_recv, void *d_packed_local, int nb, void *stream)
{
    int rc = slab_check(p, d_packed_local, nullptr, false, nb);
    if (rc) return rc;
    if (d_recv && (uintptr_t)d_recv % 16) return FFTB_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    fftb_plan zp = p->zp;
    unsigned char *A = zp->d_mem + zp->o_ws;
    const int r = p->rank, R = p->world;
    const long long n_r = p->stick_lo[r + 1] - p->stick_lo[r], pitch_r = zp->pitch;
    if (d_recv) { // [peer][band][the peer's planes][own sticks] -> A[band][all planes][own sticks]
        SlabSegs sg;
        sg.n = R;
        long long off = 0;
        int max_rows = 1;
        for (int s = 0; s < R; ++s) {
            const long long slab_s = p->z_lo[s + 1] - p->z_lo[s];
            SlabSeg &g = sg.s[s];
            g.rows = (int)slab_s; g.cols = (int)n_r; g.peer = s;
            g.src_off = off; g.src_sb = slab_s * n_r; g.src_sr = n_r;
            sg.dst[s] = A;
            g.dst_off = p->z_lo[s] * pitch_r; g.dst_sb = (long long)p->n3 * pitch_r; g.dst_sr = pitch_r;
            off += (long long)nb * slab_s * n_r;
            if (g.rows > max_rows) max_rows = g.rows;
        }
        rc = slab_copy(p, sg, d_recv, max_rows, nb, st);
        if (rc) return rc;
    }
    rc = zp->zl.fwd(zp->dev, A, d_packed_local, zp->a_fwd_stride, nb, 0, st);
    if (rc) zp->sticky = rc;
    return rc;
}

int fftb_slab_plan_destroy(fftb_slab_plan p)
{
    if (!p) return FFTB_EINVAL;
    if (p->zp) fftb_plan_destroy(p->zp);
    if (p->pp) fftb_plan_destroy(p->pp);
    delete p;
    return FFTB_OK;
}

} // extern "C"

