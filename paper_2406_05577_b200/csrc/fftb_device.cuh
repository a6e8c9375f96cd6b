// fftb_device.cuh -- complex helpers and in-register DFT codelets (sm_100a).
//
// The 1D DFT is y = DFT_n x with DFT_n = [w_n^{lk}], w_n = exp(-j 2 pi / n) (PAPER.md:48-56,
// Eq. 2-3); SIGN = -1 is that forward transform, SIGN = +1 the inverse exp(+j g r) of the
// plane-wave expansion (Eq. 8).  A codelet transforms P values held in the
// registers of ONE thread, fully unrolled, with compile-time twiddles; the Cooley-Tukey
// factorisation n = n0 x n1 is applied recursively as a radix-2 decimation in
// time down to P = 1 or P = 3, so P in {2,4,8,16} and {3,6,12} are available.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace fftb {

template <typename T> struct Cx;
template <> struct Cx<double> { using type = double2; };
template <> struct Cx<float> { using type = float2; };
template <typename T> using cx = typename Cx<T>::type;

template <typename T> __device__ __forceinline__ cx<T> mk(T re, T im) { cx<T> r; r.x = re; r.y = im; return r; }
template <typename C> __device__ __forceinline__ C cadd(C a, C b) { a.x += b.x; a.y += b.y; return a; }
template <typename C> __device__ __forceinline__ C csub(C a, C b) { a.x -= b.x; a.y -= b.y; return a; }
template <typename C> __device__ __forceinline__ C cmul(C a, C b)
{
    C r;
    r.x = a.x * b.x - a.y * b.y;
    r.y = a.x * b.y + a.y * b.x;
    return r;
}
// a * conj(b)
template <typename C> __device__ __forceinline__ C cmulc(C a, C b)
{
    C r;
    r.x = a.x * b.x + a.y * b.y;
    r.y = a.y * b.x - a.x * b.y;
    return r;
}
// multiply by w or conj(w) depending on the transform direction: tables hold exp(+j 2 pi i/N)
template <int SIGN, typename C> __device__ __forceinline__ C cmul_dir(C a, C w)
{
    if constexpr (SIGN > 0) return cmul(a, w);
    else return cmulc(a, w);
}
// multiply by j^p, p taken mod 4 (runtime): 1, j, -1, -j
template <typename C> __device__ __forceinline__ C mul_jpow(C a, int p)
{
    C r;
    const bool sw = p & 1;
    const bool ng_re = ((p + 1) & 2) != 0; // p = 1,2 -> negate the new real part
    const bool ng_im = (p & 2) != 0;       // p = 2,3 -> negate the new imaginary part
    r.x = sw ? a.y : a.x;
    r.y = sw ? a.x : a.y;
    r.x = ng_re ? -r.x : r.x;
    r.y = ng_im ? -r.y : r.y;
    return r;
}

// cos / sin of 2 pi q / 96, q in [0, 96): every root of order 2, 3, 4, 6, 8, 12, 16, 24, 32, 48 the
// codelets and the pre-/post-twiddles need, as correctly rounded literals
__host__ __device__ constexpr double cos96_first(int q)
{
    return q == 0 ? 1.0
         : q == 1 ? 0.9978589232386035067380698
         : q == 2 ? 0.9914448613738104111445575
         : q == 3 ? 0.9807852804032304491261822
         : q == 4 ? 0.9659258262890682867497432
         : q == 5 ? 0.9469301294951056642558043
         : q == 6 ? 0.9238795325112867561281832
         : q == 7 ? 0.8968727415326883038941039
         : q == 8 ? 0.8660254037844386467637232
         : q == 9 ? 0.8314696123025452370787884
         : q == 10 ? 0.793353340291235164579777
         : q == 11 ? 0.7518398074789773964075194
         : q == 12 ? 0.7071067811865475244008444
         : q == 13 ? 0.6593458151000688684251246
         : q == 14 ? 0.6087614290087206394160975
         : q == 15 ? 0.5555702330196022247428308
         : q == 16 ? 0.5
         : q == 17 ? 0.442288690219001281995239
         : q == 18 ? 0.38268343236508977172846
         : q == 19 ? 0.3214394653031615807010576
         : q == 20 ? 0.2588190451025207623488988
         : q == 21 ? 0.1950903220161282678482849
         : q == 22 ? 0.1305261922200515915484062
         : q == 23 ? 0.06540312923014306681531556
         : 0.0;
}
__host__ __device__ constexpr double cos96(int q)
{
    q = ((q % 96) + 96) % 96;
    return q <= 24 ? cos96_first(q) : q <= 48 ? -cos96_first(48 - q) : q <= 72 ? -cos96_first(q - 48) : cos96_first(96 - q);
}
__host__ __device__ constexpr double sin96(int q) { return cos96(q - 24); }

// a * exp(SIGN j 2 pi K / P), K and P compile-time
template <int K, int P, int SIGN, typename T> __device__ __forceinline__ cx<T> mul_root(cx<T> a)
{
    static_assert(96 % P == 0, "root order must divide 96");
    constexpr int q = ((K * (96 / P)) % 96 + 96) % 96;
    if constexpr (q == 0) return a;
    else if constexpr (q == 48) return mk<T>(-a.x, -a.y);
    else if constexpr (q == 24) return SIGN > 0 ? mk<T>(-a.y, a.x) : mk<T>(a.y, -a.x);
    else if constexpr (q == 72) return SIGN > 0 ? mk<T>(a.y, -a.x) : mk<T>(-a.y, a.x);
    else {
        constexpr T c = (T)cos96(q);
        constexpr T s = (T)(SIGN * sin96(q));
        return mk<T>(a.x * c - a.y * s, a.x * s + a.y * c);
    }
}

// radix-2 decimation-in-time recombination, unrolled over K at compile time
template <int K, int P, int SIGN, typename T>
__device__ __forceinline__ void dit_combine(cx<T> (&v)[P], const cx<T> (&e)[P / 2], const cx<T> (&o)[P / 2])
{
    if constexpr (K < P / 2) {
        cx<T> t = mul_root<K, P, SIGN, T>(o[K]);
        v[K] = cadd(e[K], t);
        v[K + P / 2] = csub(e[K], t);
        dit_combine<K + 1, P, SIGN, T>(v, e, o);
    }
}

// In-register DFT of length P, natural order in and out.
template <int P, int SIGN, typename T> __device__ __forceinline__ void fft_reg(cx<T> (&v)[P])
{
    using C = cx<T>;
    if constexpr (P == 1) {
        return;
    } else if constexpr (P == 3) {
        constexpr T h = (T)0.5;
        constexpr T s3 = (T)(SIGN * 0.8660254037844386467637232);
        C t1 = cadd(v[1], v[2]);
        C t2 = mk<T>(v[0].x - h * t1.x, v[0].y - h * t1.y);
        C d = csub(v[1], v[2]);
        C t3 = mk<T>(-s3 * d.y, s3 * d.x); // j * s3 * d
        v[0] = cadd(v[0], t1);
        v[1] = cadd(t2, t3);
        v[2] = csub(t2, t3);
    } else {
        static_assert(P % 2 == 0, "unsupported codelet length");
        constexpr int H = P / 2;
        C e[H], o[H];
#pragma unroll
        for (int k = 0; k < H; ++k) { e[k] = v[2 * k]; o[k] = v[2 * k + 1]; }
        fft_reg<H, SIGN, T>(e);
        fft_reg<H, SIGN, T>(o);
        // y[k] = E[k] + w_P^k O[k], y[k+H] = E[k] - w_P^k O[k]
        dit_combine<0, P, SIGN, T>(v, e, o);
    }
}

// non-negative remainder, N compile-time
template <int N> __device__ __forceinline__ int modn(int x)
{
    if constexpr ((N & (N - 1)) == 0) return x & (N - 1);
    else { int r = x % N; return r < 0 ? r + N : r; }
}

// 16-byte / 8-byte global accesses with cache hints
template <typename C> __device__ __forceinline__ C ldg_stream(const C *p) { return __ldcs(p); }
template <typename C> __device__ __forceinline__ void stg_stream(C *p, C v) { __stcs(p, v); }

// 2-element (x = 2n', 2n'+1) global accesses: 32 bytes for complex128, 16 for complex64
__device__ __forceinline__ void st_pair(double2 *p, double2 a, double2 b)
{
    asm volatile("st.global.cs.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(a.x), "d"(a.y), "d"(b.x), "d"(b.y) : "memory");
}
__device__ __forceinline__ void st_pair(float2 *p, float2 a, float2 b)
{
    __stcs(reinterpret_cast<float4 *>(p), make_float4(a.x, a.y, b.x, b.y));
}
__device__ __forceinline__ void ld_pair(const double2 *p, double2 &a, double2 &b)
{
    asm volatile("ld.global.cs.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(a.x), "=d"(a.y), "=d"(b.x), "=d"(b.y) : "l"(p));
}
__device__ __forceinline__ void ld_pair(const float2 *p, float2 &a, float2 &b)
{
    const float4 v = __ldcs(reinterpret_cast<const float4 *>(p));
    a = make_float2(v.x, v.y);
    b = make_float2(v.z, v.w);
}

// ---- L2 eviction priorities (createpolicy + .L2::cache_hint) ------------------------------------------------------
// L2 eviction priority of a global access (createpolicy): the ring of intermediate rows is kept (evict_last) while
// the cuboid and packed streams pass through (evict_first)
__device__ __forceinline__ unsigned long long l2_policy(int kind) // 0 normal, 1 evict_first, 2 evict_last
{
    unsigned long long p;
    if (kind == 2) asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    else if (kind == 1) asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    else asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ void st_pair_hint(double2 *p, double2 a, double2 b, unsigned long long pol)
{
    asm volatile("st.global.L2::cache_hint.v4.f64 [%0], {%1, %2, %3, %4}, %5;" ::"l"(p), "d"(a.x), "d"(a.y), "d"(b.x), "d"(b.y), "l"(pol) : "memory");
}
__device__ __forceinline__ void st_pair_hint(float2 *p, float2 a, float2 b, unsigned long long pol)
{
    asm volatile("st.global.L2::cache_hint.v4.f32 [%0], {%1, %2, %3, %4}, %5;" ::"l"(p), "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y), "l"(pol) : "memory");
}
__device__ __forceinline__ void st_hint(double2 *p, double2 a, unsigned long long pol)
{
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1, %2}, %3;" ::"l"(p), "d"(a.x), "d"(a.y), "l"(pol) : "memory");
}
__device__ __forceinline__ void st_hint(float2 *p, float2 a, unsigned long long pol)
{
    asm volatile("st.global.L2::cache_hint.v2.f32 [%0], {%1, %2}, %3;" ::"l"(p), "f"(a.x), "f"(a.y), "l"(pol) : "memory");
}

__device__ __forceinline__ double2 ld_hint(const double2 *p, unsigned long long pol)
{
    double2 v;
    asm volatile("ld.global.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ float2 ld_hint(const float2 *p, unsigned long long pol)
{
    float2 v;
    asm volatile("ld.global.L2::cache_hint.v2.f32 {%0, %1}, [%2], %3;" : "=f"(v.x), "=f"(v.y) : "l"(p), "l"(pol));
    return v;
}

} // namespace fftb
