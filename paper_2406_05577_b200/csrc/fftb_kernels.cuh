// fftb_kernels.cuh -- the pass kernels of the pruned sphere <-> cuboid transform (sm_100a).
//
// Pipeline (Fig. 3 and :112, "the zero-padding can be done in stages ... fuse the 1D
// transforms with the padding operations", axis order z -> y -> x as BASELINE.json's north_star fixes):
//
//   inverse  zpass_inv : packed sticks --unpack + pad + z-DFT--> A[b][z][stick]     (n_sticks lines)
//            plane     : A[b][z][.]    --pad + y-DFT on the occupied x columns, on-chip transpose,
//                                        pad + x-DFT--> cuboid[b][z][y][x]          (one z-plane per CTA group)
//   forward  plane     : cuboid        --x-DFT keeping the occupied k1, y-DFT keeping the stick rows--> A
//            zpass_fwd : A             --z-DFT keeping the stick's k3 range, scale, pack--> packed
//   vloc     plane in VLOC mode: inverse y,x passes, V(r) multiply in registers, forward x,y passes;
//            the cuboid is never written.
//
// The paper's pack/rotate codelets + MPI all-to-all between stages become the
// on-chip exchanges inside each kernel and the plane-major intermediate A, which is sized to
// stay in the 126 MB L2 between the two kernels of a band chunk.
//
// One 1D DFT of length N is split as N = R * M (decimation in frequency on the inverse side,
// decimation in time on the forward side) with M = P1 * P2 done as two in-register codelet stages
// around one shared-memory exchange:
//     inverse:  u_r[k] = sum_j x'[k + j M] w_N^{r (k + j M)}          (zero terms skipped: pruning)
//               out[R n' + r] = mu(n) * DFT_M(u_r)[n']
//     forward:  v_r[n'] = mu(n) in[R n' + r],  G_r = DFT_M(v_r)
//               out[k'] = sum_r w_N^{r k'} G_r[k' mod M]              (only k' inside the cut-off)
// x' is the input shifted by N/4 (k' = k + N/4) on a half-band axis (all data in k' in [0, N/2]),
// which makes mu(n) = (-/+ j)^n; with R = 2 the first radix-2 stage of a half-band axis costs no
// additions at all.  For the y axis the R residues are spread over R CTAs, which is what lets a
// z-plane be processed in R independent pieces that each fit in shared memory.
#pragma once
#include "fftb_device.cuh"

namespace fftb {

enum PlaneMode { MODE_INV = 0, MODE_FWD = 1, MODE_VLOC = 2 };

struct DevPlan {
    int n1, n2, n3;
    int nsticks, pitch, nxocc;
    int k1lo;          // signed k1 of x column 0
    int ry;            // number of y residues = partial A planes written by the forward plane kernel
    const int4 *stick; // {off, k3lo, len, (k1 & 0xffff) | (k2 << 16)}
    const int4 *col;   // {first stick, stick count, k2lo, 0}
    const int *colperm; // x columns with more than one stick first, then the single-stick ones
    int n_multi;       // number of multi-stick columns
    const void *tw1, *tw2, *tw3; // exp(+j 2 pi i / N_d), i < N_d, in the plan's precision
    long long S;       // points per band
    double scale;      // applied in zpass_fwd
    int sms;           // host side only: SM count of the device the plan was bound on
};

template <int N_, int R_, int P1_, int P2_, bool HALF_> struct Axis {
    static constexpr int N = N_, R = R_, P1 = P1_, P2 = P2_, M = N_ / R_;
    static constexpr bool HALF = HALF_;
    static constexpr int SH = HALF_ ? N_ / 4 : 0;           // k' = k + SH
    static constexpr int JMAX = HALF_ ? (R_ / 2 + 1) : R_;  // terms of the R-way split that can be non-zero
    static_assert(P1_ * P2_ * R_ == N_, "bad factorisation");
    static_assert(!HALF_ || (R_ % 2 == 0 && N_ % 4 == 0), "half-band axis needs an even split");
};

// element index of primed frequency kp inside a run that starts at signed frequency lo; >= cnt means "zero"
template <class AX> __device__ __forceinline__ int elem_of(int kp, int lo) { return modn<AX::N>(kp - AX::SH - lo); }

// power of j of the shift modulation mu(n): inverse exp(-2 pi j SH n / N) = (-j)^n, forward (+j)^n
template <class AX, int SIGN> __device__ __forceinline__ int mu_pow(int n)
{
    if constexpr (!AX::HALF) return 0;
    else return SIGN > 0 ? (-n) & 3 : n & 3;
}

template <typename T> __device__ __forceinline__ cx<T> czero() { return mk<T>((T)0, (T)0); }

// ---------------------------------------------------------------------------------------------
// z pass, inverse: packed -> A[b][z][stick]
// CTA = LINES consecutive sticks of one band.
// ---------------------------------------------------------------------------------------------
template <typename T, class AZ, int LINES, int NT>
__global__ void __launch_bounds__(NT) zpass_inv_k(DevPlan pl, const cx<T> *__restrict__ packed, cx<T> *__restrict__ A,
                                                  long long a_band_stride)
{
    using C = cx<T>;
    constexpr int N = AZ::N, R = AZ::R, P1 = AZ::P1, P2 = AZ::P2, M = AZ::M;
    constexpr int LP = LINES | 1;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C *exch = reinterpret_cast<C *>(smem_raw); // [M][LP]
    C *tw = exch + M * LP;                     // [N]
    const int tid = threadIdx.x;
    for (int i = tid; i < N; i += NT) tw[i] = reinterpret_cast<const C *>(pl.tw3)[i];
    const int s0 = blockIdx.x * LINES;
    const C *src = packed + (long long)blockIdx.y * pl.S;
    C *dst = A + (long long)blockIdx.y * a_band_stride;
#pragma unroll 1
    for (int r = 0; r < R; ++r) {
        __syncthreads();
        for (int task = tid; task < LINES * P2; task += NT) {
            const int l = task / P2, t = task % P2, s = s0 + l;
            if (s < pl.nsticks) {
                const int4 st = pl.stick[s];
                C x[P1];
#pragma unroll
                for (int j = 0; j < P1; ++j) {
                    const int k = t + P2 * j;
                    C acc = czero<T>();
#pragma unroll
                    for (int jj = 0; jj < AZ::JMAX; ++jj) {
                        const int kp = k + jj * M;
                        const int e = elem_of<AZ>(kp, st.y);
                        if (e < st.z) {
                            C v = src[st.x + e];
                            if (r != 0) v = cmul(v, tw[modn<N>(r * kp)]);
                            acc = cadd(acc, v);
                        }
                    }
                    x[j] = acc;
                }
                fft_reg<P1, +1, T>(x);
#pragma unroll
                for (int m = 0; m < P1; ++m) {
                    C v = x[m];
                    if (m != 0) v = cmul(v, tw[modn<N>(t * m * R)]);
                    exch[(m * P2 + t) * LP + l] = v;
                }
            }
        }
        __syncthreads();
        for (int task = tid; task < LINES * P1; task += NT) {
            const int m = task / LINES, l = task % LINES, s = s0 + l;
            if (s < pl.nsticks) {
                C y[P2];
#pragma unroll
                for (int t = 0; t < P2; ++t) y[t] = exch[(m * P2 + t) * LP + l];
                fft_reg<P2, +1, T>(y);
#pragma unroll
                for (int q = 0; q < P2; ++q) {
                    const int n = R * (m + P1 * q) + r;
                    dst[(long long)n * pl.pitch + s] = mul_jpow(y[q], mu_pow<AZ, +1>(n));
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// z pass, forward: A (sum of the ry partial planes) -> packed, scaled
// ---------------------------------------------------------------------------------------------
template <typename T, class AZ, int LINES, int NT>
__global__ void __launch_bounds__(NT) zpass_fwd_k(DevPlan pl, const cx<T> *__restrict__ A, cx<T> *__restrict__ packed,
                                                  long long a_band_stride)
{
    using C = cx<T>;
    // forward uses the transposed factorisation: stage 1 radix P2 over j, stage 2 radix P1 over t
    constexpr int N = AZ::N, R = AZ::R, Q1 = AZ::P2, Q2 = AZ::P1, M = AZ::M;
    constexpr int LP = LINES | 1;
    constexpr int MP = Q2 * LP + 1; // pitch between stage-1 output indices m (odd: conflict-free for lanes over m)
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C *exch = reinterpret_cast<C *>(smem_raw); // [R][Q1][MP]
    C *tw = exch + R * Q1 * MP;                // [N]
    const int tid = threadIdx.x;
    for (int i = tid; i < N; i += NT) tw[i] = reinterpret_cast<const C *>(pl.tw3)[i];
    const int s0 = blockIdx.x * LINES;
    const C *src = A + (long long)blockIdx.y * a_band_stride;
    C *dst = packed + (long long)blockIdx.y * pl.S;
    const long long rstride = (long long)pl.n3 * pl.pitch; // between partial planes
    const T scale = (T)pl.scale;
    __syncthreads();
    // stage 1: task (t, l), lanes over l (coalesced reads of A)
    for (int task = tid; task < LINES * Q2; task += NT) {
        const int t = task / LINES, l = task % LINES, s = s0 + l;
        if (s < pl.nsticks) {
#pragma unroll
            for (int r = 0; r < R; ++r) {
                C x[Q1];
#pragma unroll
                for (int j = 0; j < Q1; ++j) {
                    const int n = R * (t + Q2 * j) + r;
                    C v = src[(long long)n * pl.pitch + s];
                    for (int p = 1; p < pl.ry; ++p) v = cadd(v, src[p * rstride + (long long)n * pl.pitch + s]);
                    x[j] = mul_jpow(v, mu_pow<AZ, -1>(n));
                }
                fft_reg<Q1, -1, T>(x);
#pragma unroll
                for (int m = 0; m < Q1; ++m) {
                    C v = x[m];
                    if (m != 0) v = cmulc(v, tw[modn<N>(t * m * R)]);
                    exch[(r * Q1 + m) * MP + t * LP + l] = v;
                }
            }
        }
    }
    __syncthreads();
    // stage 2: task (l, m), lanes over m (coalesced writes of the stick)
    for (int task = tid; task < LINES * Q1; task += NT) {
        const int l = task / Q1, m = task % Q1, s = s0 + l;
        if (s < pl.nsticks) {
            const int4 st = pl.stick[s];
            C g[R][Q2];
#pragma unroll
            for (int r = 0; r < R; ++r) {
#pragma unroll
                for (int t = 0; t < Q2; ++t) g[r][t] = exch[(r * Q1 + m) * MP + t * LP + l];
                fft_reg<Q2, -1, T>(g[r]);
            }
#pragma unroll
            for (int q = 0; q < Q2; ++q) {
                const int kk = m + Q1 * q; // output index of the length-M transforms
#pragma unroll
                for (int jj = 0; jj < AZ::JMAX; ++jj) {
                    const int kp = kk + jj * M;
                    const int e = elem_of<AZ>(kp, st.y);
                    if (e < st.z) {
                        C acc = g[0][q];
#pragma unroll
                        for (int r = 1; r < R; ++r) acc = cadd(acc, cmulc(g[r][q], tw[modn<N>(r * kp)]));
                        dst[st.x + e] = mk<T>(acc.x * scale, acc.y * scale);
                    }
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// plane kernel: the y and x passes of one z-plane, one y residue class per CTA
//   grid = (ry * n3, bands);  blockIdx.x = z * ry + r
// ---------------------------------------------------------------------------------------------
template <typename T, class AX, class AY, int LX, int LY, int NT> struct PlaneSmem {
    using C = cx<T>;
    static constexpr int MY = AY::M;                // y lines per CTA
    static constexpr int YP = MY | 1;               // pitch of one x column in the plane buffer
    static constexpr int NCOL = AX::HALF ? AX::N / 2 + 1 : AX::N;
    static constexpr int LXP = LX | 1;
    // x exchange: [M1 values][LX lines], one extra element per stage-1 output index group
    static constexpr int XMP = AX::P2 * LXP + 1;    // inverse: pitch between m (lanes over m in stage 2)
    static constexpr int XFP = AX::P1 * LXP + 1;    // forward (transposed factorisation)
    static constexpr int XEX = (AX::P1 * XMP > AX::P2 * XFP ? AX::P1 * XMP : AX::P2 * XFP);
    static constexpr int P2YP = AY::P2 + 1;         // y exchange pitch (odd)
    static constexpr int YEXI = LY * AY::P1 * P2YP, YEXF = LY * AY::P2 * (AY::P1 + 1);
    static constexpr int YEX = (YEXI > YEXF ? YEXI : YEXF);
    static constexpr int EX = (XEX > YEX ? XEX : YEX);
    static constexpr size_t bytes = sizeof(C) * ((size_t)NCOL * YP + EX + AX::N + AY::N);
};

template <typename T, class AX, class AY, int LX, int LY, int NT, int MODE>
__global__ void __launch_bounds__(NT) plane_k(DevPlan pl, const cx<T> *__restrict__ Ain, cx<T> *__restrict__ Aout,
                                              const cx<T> *__restrict__ cub_in, cx<T> *__restrict__ cub_out,
                                              const T *__restrict__ vloc, long long a_in_stride, long long a_out_stride)
{
    using C = cx<T>;
    using SM = PlaneSmem<T, AX, AY, LX, LY, NT>;
    constexpr int N1 = AX::N, RX = AX::R, P1 = AX::P1, P2 = AX::P2, M1 = AX::M;
    constexpr int N2 = AY::N, RY = AY::R, PY1 = AY::P1, PY2 = AY::P2, MY = AY::M;
    constexpr int YP = SM::YP, LXP = SM::LXP;
    static_assert(MY % LX == 0, "LX must divide the lines per CTA");
    static_assert(LX * P1 <= NT && LX * P2 <= NT, "x stages are one task per thread");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C *pbuf = reinterpret_cast<C *>(smem_raw); // plane buffer [NCOL][YP]: column c, local line y'
    C *exch = pbuf + SM::NCOL * YP;
    C *tw1 = exch + SM::EX;
    C *tw2 = tw1 + N1;
    const int tid = threadIdx.x;
    const int z = blockIdx.x / RY, ry = blockIdx.x % RY, b = blockIdx.y;
    for (int i = tid; i < N1; i += NT) tw1[i] = reinterpret_cast<const C *>(pl.tw1)[i];
    for (int i = tid; i < N2; i += NT) tw2[i] = reinterpret_cast<const C *>(pl.tw2)[i];
    const int nx = pl.nxocc;

    // ------------------------------------------------------------------ inverse y pass -> pbuf
    if constexpr (MODE != MODE_FWD) {
        const C *src = Ain + (long long)b * a_in_stride + (long long)z * pl.pitch;
        C *ex = exch; // [LY][PY1][P2YP]
        for (int c0 = 0; c0 < nx; c0 += LY) {
            __syncthreads();
            for (int task = tid; task < LY * PY2; task += NT) {
                const int cl = task / PY2, t = task % PY2, c = c0 + cl;
                if (c < nx) {
                    const int4 co = pl.col[c];
                    C x[PY1];
#pragma unroll
                    for (int j = 0; j < PY1; ++j) {
                        const int k = t + PY2 * j;
                        C acc = czero<T>();
#pragma unroll
                        for (int jj = 0; jj < AY::JMAX; ++jj) {
                            const int kp = k + jj * MY;
                            const int e = elem_of<AY>(kp, co.z);
                            if (e < co.y) {
                                C v = src[co.x + e];
                                if (ry != 0) v = cmul(v, tw2[modn<N2>(ry * kp)]);
                                acc = cadd(acc, v);
                            }
                        }
                        x[j] = acc;
                    }
                    fft_reg<PY1, +1, T>(x);
#pragma unroll
                    for (int m = 0; m < PY1; ++m) {
                        C v = x[m];
                        if (m != 0) v = cmul(v, tw2[modn<N2>(t * m * RY)]);
                        ex[(cl * PY1 + m) * SM::P2YP + t] = v;
                    }
                }
            }
            __syncthreads();
            for (int task = tid; task < LY * PY1; task += NT) {
                const int cl = task / PY1, m = task % PY1, c = c0 + cl;
                if (c < nx) {
                    C y[PY2];
#pragma unroll
                    for (int t = 0; t < PY2; ++t) y[t] = ex[(cl * PY1 + m) * SM::P2YP + t];
                    fft_reg<PY2, +1, T>(y);
#pragma unroll
                    for (int q = 0; q < PY2; ++q) {
                        const int yl = m + PY1 * q;
                        pbuf[c * YP + yl] = mul_jpow(y[q], mu_pow<AY, +1>(RY * yl + ry));
                    }
                }
            }
        }
    }

    // ------------------------------------------------------------------ x passes, LX lines at a time
    for (int y0 = 0; y0 < MY; y0 += LX) {
        C reg[RX][P2]; // the line values x = RX (m + P1 q) + e held by thread (line, m)
        const int ml = tid % P1, yl2 = tid / P1; // stage-2 (inverse) / stage-1 (forward) role: lanes over m
        const bool act2 = tid < LX * P1;
        const int ygl = RY * (y0 + yl2) + ry;     // global y of that role's line
        if constexpr (MODE != MODE_FWD) {
            // inverse x: stage 1, thread (t, line) with lanes over lines
            const int t = tid / LX, yl = tid % LX;
#pragma unroll
            for (int e = 0; e < RX; ++e) {
                __syncthreads(); // pbuf complete / exch free
                if (tid < LX * P2) {
                    C x[P1];
#pragma unroll
                    for (int j = 0; j < P1; ++j) {
                        const int k = t + P2 * j;
                        C acc = czero<T>();
#pragma unroll
                        for (int jj = 0; jj < AX::JMAX; ++jj) {
                            const int kp = k + jj * M1;
                            const int c = elem_of<AX>(kp, pl.k1lo);
                            if (c < nx) {
                                C v = pbuf[c * YP + y0 + yl];
                                if (e != 0) v = cmul(v, tw1[modn<N1>(e * kp)]);
                                acc = cadd(acc, v);
                            }
                        }
                        x[j] = acc;
                    }
                    fft_reg<P1, +1, T>(x);
#pragma unroll
                    for (int m = 0; m < P1; ++m) {
                        C v = x[m];
                        if (m != 0) v = cmul(v, tw1[modn<N1>(t * m * RX)]);
                        exch[m * SM::XMP + t * LXP + yl] = v;
                    }
                }
                __syncthreads();
                if (act2) {
                    C y[P2];
#pragma unroll
                    for (int tt = 0; tt < P2; ++tt) y[tt] = exch[ml * SM::XMP + tt * LXP + yl2];
                    fft_reg<P2, +1, T>(y);
#pragma unroll
                    for (int q = 0; q < P2; ++q) {
                        const int n = RX * (ml + P1 * q) + e;
                        reg[e][q] = mul_jpow(y[q], mu_pow<AX, +1>(n));
                    }
                }
            }
            if constexpr (MODE == MODE_INV) {
                if (act2) {
                    C *row = cub_out + (((long long)b * pl.n3 + z) * N2 + ygl) * N1;
#pragma unroll
                    for (int q = 0; q < P2; ++q) {
                        if constexpr (RX == 2) st_pair(row + 2 * (ml + P1 * q), reg[0][q], reg[1][q]); // one 32-byte store
                        else {
#pragma unroll
                            for (int e = 0; e < RX; ++e) stg_stream(row + RX * (ml + P1 * q) + e, reg[e][q]);
                        }
                    }
                }
            }
        }
        if constexpr (MODE == MODE_VLOC) {
            if (act2) {
                const T *vrow = vloc + ((long long)z * N2 + ygl) * N1;
#pragma unroll
                for (int q = 0; q < P2; ++q)
#pragma unroll
                    for (int e = 0; e < RX; ++e) {
                        const T v = vrow[RX * (ml + P1 * q) + e];
                        reg[e][q].x *= v;
                        reg[e][q].y *= v;
                    }
            }
        }
        if constexpr (MODE == MODE_FWD) {
            if (act2) {
                const C *row = cub_in + (((long long)b * pl.n3 + z) * N2 + ygl) * N1;
#pragma unroll
                for (int q = 0; q < P2; ++q) {
                    if constexpr (RX == 2) ld_pair(row + 2 * (ml + P1 * q), reg[0][q], reg[1][q]);
                    else {
#pragma unroll
                        for (int e = 0; e < RX; ++e) reg[e][q] = ldg_stream(row + RX * (ml + P1 * q) + e);
                    }
                }
            }
        }
        if constexpr (MODE != MODE_INV) {
            // forward x (transposed factorisation): stage 1 radix P2 over q by thread (line, t = ml),
            // stage 2 radix P1 over t by thread (m', line) with lanes over lines
            C g[RX][P1];
            const int mq = tid / LX, yl = tid % LX;
            const bool act1 = tid < LX * P2;
#pragma unroll
            for (int e = 0; e < RX; ++e) {
                __syncthreads(); // exch free (also orders the inverse stage-2 reads before these writes)
                if (act2) {
                    C x[P2];
#pragma unroll
                    for (int q = 0; q < P2; ++q) {
                        const int n = RX * (ml + P1 * q) + e;
                        x[q] = mul_jpow(reg[e][q], mu_pow<AX, -1>(n));
                    }
                    fft_reg<P2, -1, T>(x);
#pragma unroll
                    for (int m = 0; m < P2; ++m) {
                        C v = x[m];
                        if (m != 0) v = cmulc(v, tw1[modn<N1>(ml * m * RX)]);
                        exch[(m * P1 + ml) * LXP + yl2] = v;
                    }
                }
                __syncthreads();
                if (act1) {
                    C y[P1];
#pragma unroll
                    for (int tt = 0; tt < P1; ++tt) y[tt] = exch[(mq * P1 + tt) * LXP + yl];
                    fft_reg<P1, -1, T>(y);
#pragma unroll
                    for (int q = 0; q < P1; ++q) g[e][q] = y[q];
                }
            }
            // combine the RX sub-transforms and keep only the occupied k1 columns -> pbuf
            // (in VLOC mode this overwrites the lines just consumed: same thread-independent footprint,
            //  but other threads' stage-1 reads of these lines finished before the last barrier)
            if (act1) {
#pragma unroll
                for (int q = 0; q < P1; ++q) {
                    const int kk = mq + P2 * q;
#pragma unroll
                    for (int jj = 0; jj < AX::JMAX; ++jj) {
                        const int kp = kk + jj * M1;
                        const int c = elem_of<AX>(kp, pl.k1lo);
                        if (c < nx) {
                            C acc = g[0][q];
#pragma unroll
                            for (int r = 1; r < RX; ++r) acc = cadd(acc, cmulc(g[r][q], tw1[modn<N1>(r * kp)]));
                            pbuf[c * YP + y0 + yl] = acc;
                        }
                    }
                }
            }
        }
    }

    // ------------------------------------------------------------------ forward y pass: pbuf -> partial A
    if constexpr (MODE != MODE_INV) {
        C *dst = Aout + (long long)b * a_out_stride + ((long long)ry * pl.n3 + z) * pl.pitch;
        // transposed factorisation: stage 1 radix PY2 over j (thread (column, t), t < PY1), stage 2 radix PY1
        constexpr int Q1 = PY2, Q2 = PY1;
        C *ex = exch; // [LY][Q1][Q2+1]
        constexpr int QP = Q2 + 1;
        for (int c0 = 0; c0 < nx; c0 += LY) {
            __syncthreads();
            for (int task = tid; task < LY * Q2; task += NT) {
                const int cl = task / Q2, t = task % Q2, c = c0 + cl;
                if (c < nx) {
                    C x[Q1];
#pragma unroll
                    for (int j = 0; j < Q1; ++j) {
                        const int yl = t + Q2 * j;
                        x[j] = mul_jpow(pbuf[c * YP + yl], mu_pow<AY, -1>(RY * yl + ry));
                    }
                    fft_reg<Q1, -1, T>(x);
#pragma unroll
                    for (int m = 0; m < Q1; ++m) {
                        C v = x[m];
                        if (m != 0) v = cmulc(v, tw2[modn<N2>(t * m * RY)]);
                        ex[(cl * Q1 + m) * QP + t] = v;
                    }
                }
            }
            __syncthreads();
            for (int task = tid; task < LY * Q1; task += NT) {
                const int cl = task / Q1, m = task % Q1, c = c0 + cl;
                if (c < nx) {
                    const int4 co = pl.col[c];
                    C y[Q2];
#pragma unroll
                    for (int t = 0; t < Q2; ++t) y[t] = ex[(cl * Q1 + m) * QP + t];
                    fft_reg<Q2, -1, T>(y);
#pragma unroll
                    for (int q = 0; q < Q2; ++q) {
                        const int kk = m + Q1 * q;
#pragma unroll
                        for (int jj = 0; jj < AY::JMAX; ++jj) {
                            const int kp = kk + jj * MY;
                            const int e = elem_of<AY>(kp, co.z);
                            if (e < co.y) {
                                C v = y[q];
                                if (ry != 0) v = cmulc(v, tw2[modn<N2>(ry * kp)]);
                                dst[co.x + e] = v;
                            }
                        }
                    }
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// dense comparison arm: scatter / gather between the pruned and the dense packed layouts
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void dense_embed_k(const int4 *__restrict__ stick, int nsticks, long long S, const cx<T> *__restrict__ src,
                              cx<T> *__restrict__ dst, int n1, int n2, int n3, bool extract)
{
    // one warp per stick
    const int warps = (blockDim.x * gridDim.x) >> 5;
    const int lane = threadIdx.x & 31;
    const long long dS = (long long)n1 * n2 * n3;
    for (int s = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; s < nsticks; s += warps) {
        const int4 st = stick[s]; // {off, k3lo, len, k1 | k2 packed}
        const int k1 = (short)(st.w & 0xffff), k2 = (short)((unsigned)st.w >> 16);
        // dense packed order: (k1 + n1/2, k2 + n2/2, k3 + n3/2), k3 fastest
        const long long base = ((long long)(k1 + n1 / 2) * n2 + (k2 + n2 / 2)) * n3 + (st.y + n3 / 2);
        for (int i = lane; i < st.z; i += 32) {
            if (extract) dst[(long long)blockIdx.y * S + st.x + i] = src[(long long)blockIdx.y * dS + base + i];
            else dst[(long long)blockIdx.y * dS + base + i] = src[(long long)blockIdx.y * S + st.x + i];
        }
    }
}

// ---------------------------------------------------------------------------------------------
// packed arrays between the paper's batch-fastest order (Fig. 8 "b x y z": element
// [point][band]) and this library's band-slowest order [band][point]: out[c][r] = in[r][c] for an
// R x Cn matrix, 32 x 32 tiles through shared memory, both sides coalesced.
// ---------------------------------------------------------------------------------------------
template <typename E>
__global__ void __launch_bounds__(256) transpose_k(const E *__restrict__ in, E *__restrict__ out, long long R, long long Cn)
{
    __shared__ E tile[32][33];
    const long long tcols = (Cn + 31) / 32; // one-dimensional grid of tiles: either side may be the long one
    const long long c0 = ((long long)blockIdx.x % tcols) * 32, r0 = ((long long)blockIdx.x / tcols) * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
#pragma unroll
    for (int i = ty; i < 32; i += 8)
        if (r0 + i < R && c0 + tx < Cn) tile[i][tx] = in[(r0 + i) * Cn + c0 + tx];
    __syncthreads();
#pragma unroll
    for (int i = ty; i < 32; i += 8)
        if (c0 + i < Cn && r0 + tx < R) out[(c0 + i) * R + r0 + tx] = tile[tx][i];
}

} // namespace fftb
