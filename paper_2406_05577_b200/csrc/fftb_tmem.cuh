// fftb_tmem.cuh -- tensor memory (TMEM) as per-thread scratch (sm_100a): 16 complex values of one thread parked in, and
// fetched from, the 32 lanes x N columns its warp may access (tcgen05.st / tcgen05.ld, shape 32x32b: thread i of the warp
// <-> TMEM lane 32 (warp % 4) + i, one 32-bit column per register).  No tensor-core arithmetic is involved: the 256 KB
// of an SM are used as a third on-chip store next to registers and shared memory.
#pragma once
#include "fftb_device.cuh"

namespace fftb {

__device__ __forceinline__ void tmem_st_x64(unsigned taddr, const unsigned (&w)[64])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x64.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32, %33, %34, %35, %36, %37, %38, %39, %40, %41, %42, %43, %44, %45, %46, %47, %48, %49, %50, %51, %52, %53, %54, %55, %56, %57, %58, %59, %60, %61, %62, %63, %64};" ::"r"(taddr), "r"(w[0]), "r"(w[1]), "r"(w[2]), "r"(w[3]), "r"(w[4]), "r"(w[5]), "r"(w[6]), "r"(w[7]), "r"(w[8]), "r"(w[9]), "r"(w[10]), "r"(w[11]), "r"(w[12]), "r"(w[13]), "r"(w[14]), "r"(w[15]), "r"(w[16]), "r"(w[17]), "r"(w[18]), "r"(w[19]), "r"(w[20]), "r"(w[21]), "r"(w[22]), "r"(w[23]), "r"(w[24]), "r"(w[25]), "r"(w[26]), "r"(w[27]), "r"(w[28]), "r"(w[29]), "r"(w[30]), "r"(w[31]), "r"(w[32]), "r"(w[33]), "r"(w[34]), "r"(w[35]), "r"(w[36]), "r"(w[37]), "r"(w[38]), "r"(w[39]), "r"(w[40]), "r"(w[41]), "r"(w[42]), "r"(w[43]), "r"(w[44]), "r"(w[45]), "r"(w[46]), "r"(w[47]), "r"(w[48]), "r"(w[49]), "r"(w[50]), "r"(w[51]), "r"(w[52]), "r"(w[53]), "r"(w[54]), "r"(w[55]), "r"(w[56]), "r"(w[57]), "r"(w[58]), "r"(w[59]), "r"(w[60]), "r"(w[61]), "r"(w[62]), "r"(w[63]) : "memory");
}
__device__ __forceinline__ void tmem_ld_x64(unsigned taddr, unsigned (&w)[64])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x64.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32, %33, %34, %35, %36, %37, %38, %39, %40, %41, %42, %43, %44, %45, %46, %47, %48, %49, %50, %51, %52, %53, %54, %55, %56, %57, %58, %59, %60, %61, %62, %63}, [%64];" : "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3]), "=r"(w[4]), "=r"(w[5]), "=r"(w[6]), "=r"(w[7]), "=r"(w[8]), "=r"(w[9]), "=r"(w[10]), "=r"(w[11]), "=r"(w[12]), "=r"(w[13]), "=r"(w[14]), "=r"(w[15]), "=r"(w[16]), "=r"(w[17]), "=r"(w[18]), "=r"(w[19]), "=r"(w[20]), "=r"(w[21]), "=r"(w[22]), "=r"(w[23]), "=r"(w[24]), "=r"(w[25]), "=r"(w[26]), "=r"(w[27]), "=r"(w[28]), "=r"(w[29]), "=r"(w[30]), "=r"(w[31]), "=r"(w[32]), "=r"(w[33]), "=r"(w[34]), "=r"(w[35]), "=r"(w[36]), "=r"(w[37]), "=r"(w[38]), "=r"(w[39]), "=r"(w[40]), "=r"(w[41]), "=r"(w[42]), "=r"(w[43]), "=r"(w[44]), "=r"(w[45]), "=r"(w[46]), "=r"(w[47]), "=r"(w[48]), "=r"(w[49]), "=r"(w[50]), "=r"(w[51]), "=r"(w[52]), "=r"(w[53]), "=r"(w[54]), "=r"(w[55]), "=r"(w[56]), "=r"(w[57]), "=r"(w[58]), "=r"(w[59]), "=r"(w[60]), "=r"(w[61]), "=r"(w[62]), "=r"(w[63]) : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_st_x32(unsigned taddr, const unsigned (&w)[32])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};" ::"r"(taddr), "r"(w[0]), "r"(w[1]), "r"(w[2]), "r"(w[3]), "r"(w[4]), "r"(w[5]), "r"(w[6]), "r"(w[7]), "r"(w[8]), "r"(w[9]), "r"(w[10]), "r"(w[11]), "r"(w[12]), "r"(w[13]), "r"(w[14]), "r"(w[15]), "r"(w[16]), "r"(w[17]), "r"(w[18]), "r"(w[19]), "r"(w[20]), "r"(w[21]), "r"(w[22]), "r"(w[23]), "r"(w[24]), "r"(w[25]), "r"(w[26]), "r"(w[27]), "r"(w[28]), "r"(w[29]), "r"(w[30]), "r"(w[31]) : "memory");
}
__device__ __forceinline__ void tmem_ld_x32(unsigned taddr, unsigned (&w)[32])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];" : "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3]), "=r"(w[4]), "=r"(w[5]), "=r"(w[6]), "=r"(w[7]), "=r"(w[8]), "=r"(w[9]), "=r"(w[10]), "=r"(w[11]), "=r"(w[12]), "=r"(w[13]), "=r"(w[14]), "=r"(w[15]), "=r"(w[16]), "=r"(w[17]), "=r"(w[18]), "=r"(w[19]), "=r"(w[20]), "=r"(w[21]), "=r"(w[22]), "=r"(w[23]), "=r"(w[24]), "=r"(w[25]), "=r"(w[26]), "=r"(w[27]), "=r"(w[28]), "=r"(w[29]), "=r"(w[30]), "=r"(w[31]) : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// one warp of the CTA allocates `cols` columns (a power of two >= 32; 512 = everything) and leaves the base address in *slot
// (shared memory); the caller then runs tmem_publish() with ALL threads of the CTA before anybody reads *slot
__device__ __forceinline__ void tmem_alloc(unsigned *slot, unsigned cols)
{
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(slot)), "r"(cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_publish()
{
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(unsigned taddr, unsigned cols)
{
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(cols) : "memory");
}

// 16 complex values <-> consecutive columns starting at taddr (64 columns for complex128, 32 for complex64)
__device__ __forceinline__ void tmem_put16(unsigned taddr, const double2 (&a)[8], const double2 (&b)[8])
{
    unsigned w[64];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        w[4 * i] = (unsigned)__double2loint(a[i].x); w[4 * i + 1] = (unsigned)__double2hiint(a[i].x);
        w[4 * i + 2] = (unsigned)__double2loint(a[i].y); w[4 * i + 3] = (unsigned)__double2hiint(a[i].y);
        w[32 + 4 * i] = (unsigned)__double2loint(b[i].x); w[32 + 4 * i + 1] = (unsigned)__double2hiint(b[i].x);
        w[32 + 4 * i + 2] = (unsigned)__double2loint(b[i].y); w[32 + 4 * i + 3] = (unsigned)__double2hiint(b[i].y);
    }
    tmem_st_x64(taddr, w);
}
__device__ __forceinline__ void tmem_put16(unsigned taddr, const float2 (&a)[8], const float2 (&b)[8])
{
    unsigned w[32];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        w[2 * i] = __float_as_uint(a[i].x); w[2 * i + 1] = __float_as_uint(a[i].y);
        w[16 + 2 * i] = __float_as_uint(b[i].x); w[16 + 2 * i + 1] = __float_as_uint(b[i].y);
    }
    tmem_st_x32(taddr, w);
}
// the loads are asynchronous: tmem_wait_ld() before the first use of the words
struct TmemWords128 { unsigned w[64]; };
struct TmemWords64 { unsigned w[32]; };
template <typename T> struct TmemWords;
template <> struct TmemWords<double> { using type = TmemWords128; };
template <> struct TmemWords<float> { using type = TmemWords64; };
__device__ __forceinline__ void tmem_get16_issue(unsigned taddr, TmemWords128 &o) { tmem_ld_x64(taddr, o.w); }
__device__ __forceinline__ void tmem_get16_issue(unsigned taddr, TmemWords64 &o) { tmem_ld_x32(taddr, o.w); }
__device__ __forceinline__ void tmem_add16(const TmemWords128 &o, double2 (&a)[8], double2 (&b)[8])
{
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        a[i].x += __hiloint2double((int)o.w[4 * i + 1], (int)o.w[4 * i]); a[i].y += __hiloint2double((int)o.w[4 * i + 3], (int)o.w[4 * i + 2]);
        b[i].x += __hiloint2double((int)o.w[32 + 4 * i + 1], (int)o.w[32 + 4 * i]); b[i].y += __hiloint2double((int)o.w[32 + 4 * i + 3], (int)o.w[32 + 4 * i + 2]);
    }
}
__device__ __forceinline__ void tmem_add16(const TmemWords64 &o, float2 (&a)[8], float2 (&b)[8])
{
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        a[i].x += __uint_as_float(o.w[2 * i]); a[i].y += __uint_as_float(o.w[2 * i + 1]);
        b[i].x += __uint_as_float(o.w[16 + 2 * i]); b[i].y += __uint_as_float(o.w[16 + 2 * i + 1]);
    }
}
__device__ __forceinline__ void tmem_unpack16(const TmemWords128 &o, double2 (&a)[8], double2 (&b)[8])
{
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        a[i].x = __hiloint2double((int)o.w[4 * i + 1], (int)o.w[4 * i]); a[i].y = __hiloint2double((int)o.w[4 * i + 3], (int)o.w[4 * i + 2]);
        b[i].x = __hiloint2double((int)o.w[32 + 4 * i + 1], (int)o.w[32 + 4 * i]); b[i].y = __hiloint2double((int)o.w[32 + 4 * i + 3], (int)o.w[32 + 4 * i + 2]);
    }
}
__device__ __forceinline__ void tmem_unpack16(const TmemWords64 &o, float2 (&a)[8], float2 (&b)[8])
{
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        a[i].x = __uint_as_float(o.w[2 * i]); a[i].y = __uint_as_float(o.w[2 * i + 1]);
        b[i].x = __uint_as_float(o.w[16 + 2 * i]); b[i].y = __uint_as_float(o.w[16 + 2 * i + 1]);
    }
}
template <typename T> __host__ __device__ constexpr int tmem_cols16() { return 16 * (int)sizeof(cx<T>) / 4; } // columns taken by 16 values

} // namespace fftb
