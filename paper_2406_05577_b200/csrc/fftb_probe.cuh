// fftb_probe.cuh -- device probe behind fftb_probe_fma: the FMA rate of the plain FP64 / FP32 pipes (sm_100a).
//
// The fused local-potential kernels never move a cuboid, so bench.py bounds them by arithmetic ("bound": "alu",
// "FP64 pipe utilisation ... over the probed peak"); MEASURED_PEAKS.json carries no ALU peak.  The
// probe is a register-only loop: every thread runs ILP independent chains of dependent FMAs, 8 warps x 4 CTAs per SM,
// nothing touches memory until one value per thread is written at the end so that the loop cannot be removed.
#pragma once
#include <cuda_runtime.h>

namespace fftb {

template <typename T, int ILP> __global__ void __launch_bounds__(256) probe_fma_k(T *out, int iters, T a, T b)
{
    T acc[ILP];
#pragma unroll
    for (int i = 0; i < ILP; ++i) acc[i] = (T)(threadIdx.x + i);
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u)
#pragma unroll
            for (int i = 0; i < ILP; ++i) acc[i] = acc[i] * a + b; // one FMA each
    }
    T s = (T)0;
#pragma unroll
    for (int i = 0; i < ILP; ++i) s += acc[i];
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// runs the probe on the current device's legacy stream and waits for it; returns TFLOP/s (2 flops per FMA) or < 0
template <typename T> double probe_fma_tflops(double *ms_out)
{
    constexpr int ILP = 8, ITERS = 4096, REPS = 5;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -1.0;
    const int grid = sms * 4;
    T *out = nullptr;
    if (cudaMalloc(&out, sizeof(T) * (size_t)grid * 256) != cudaSuccess) return -1.0;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    double best = 1e30;
    for (int r = 0; r < REPS + 1; ++r) { // the first run warms up
        cudaEventRecord(e0, 0);
        probe_fma_k<T, ILP><<<grid, 256>>>(out, ITERS, (T)0.999999, (T)1e-6);
        cudaEventRecord(e1, 0);
        if (cudaEventSynchronize(e1) != cudaSuccess) { best = -1.0; break; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (r > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    if (best <= 0.0 || cudaGetLastError() != cudaSuccess) return -1.0;
    if (ms_out) *ms_out = best;
    const double fma = (double)grid * 256.0 * ITERS * 8.0 * ILP;
    return 2.0 * fma / (best * 1e-3) / 1e12;
}

// ---- store port: how many bytes per clock ONE SM can push to global memory -------------------------------------------
// The inverse plane kernels issue a z-plane's 262 KB of cuboid stores within their x phase; this probe shows the rate an
// SM cannot exceed however few SMs are storing (32 B/clk on B200), which is what bounds that phase.
__global__ void __launch_bounds__(256, 1) probe_store_k(double2 *out, long long per_cta_elems, int iters, long long *clk)
{
    double2 *base = out + (long long)blockIdx.x * per_cta_elems;
    const int tid = threadIdx.x;
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
        // every warp writes 1 KB per instruction (32 lanes x 32 B), 16 instructions back to back like an x task
        double2 *p = base + ((long long)it * 256 * 16 + tid) * 2;
#pragma unroll
        for (int u = 0; u < 16; ++u)
            asm volatile("st.global.cs.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p + (long long)u * 512), "d"(1.0), "d"(2.0), "d"(3.0), "d"((double)it) : "memory");
    }
    __syncthreads();
    if (tid == 0) clk[blockIdx.x] = clock64() - t0;
}

// n_ctas CTAs (one per SM) stream 32 MB each; returns bytes per clock per SM (issue-side clocks), aggregate GB/s in *gbs
inline double probe_store_port(int n_ctas, double *gbs)
{
    constexpr int ITERS = 256;
    const long long per_cta = (long long)ITERS * 256 * 16 * 2;
    double2 *out = nullptr;
    long long *clk = nullptr;
    if (n_ctas < 1 || cudaMalloc(&out, sizeof(double2) * (size_t)per_cta * n_ctas) != cudaSuccess) return -1.0;
    if (cudaMalloc(&clk, sizeof(long long) * (size_t)n_ctas) != cudaSuccess) { cudaFree(out); return -1.0; }
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    probe_store_k<<<n_ctas, 256>>>(out, per_cta, 8, clk); // warm-up
    cudaEventRecord(e0, 0);
    probe_store_k<<<n_ctas, 256>>>(out, per_cta, ITERS, clk);
    cudaEventRecord(e1, 0);
    double res = -1.0;
    if (cudaEventSynchronize(e1) == cudaSuccess && cudaGetLastError() == cudaSuccess) {
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        long long *h = new long long[n_ctas];
        cudaMemcpy(h, clk, sizeof(long long) * (size_t)n_ctas, cudaMemcpyDeviceToHost);
        double avg = 0.0;
        for (int i = 0; i < n_ctas; ++i) avg += (double)h[i];
        delete[] h;
        const double bytes = (double)per_cta * 16.0;
        res = bytes / (avg / n_ctas);
        if (gbs) *gbs = bytes * n_ctas / (ms * 1e-3) / 1e9;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    cudaFree(clk);
    return res;
}

} // namespace fftb
