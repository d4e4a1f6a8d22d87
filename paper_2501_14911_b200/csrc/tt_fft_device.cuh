// tt_fft_device.cuh - device-side building blocks of the batched mixed-radix FFTs along time (tt_fft.cu) shared with the
// fused adjoint kernel (tt_gemv.cu): compile-time trigonometry, register butterflies, the decimation-in-frequency passes
// over a shared-memory tile sm[n*T + t] (series index fastest), and the real-output store of the inverse transform.
// See the header of tt_fft.cu for the algorithm.
#pragma once
#include <type_traits>

#include "tt_common.cuh"
#include "tt_internal.h"

namespace tt {

// ---------------------------------------------------------------------------------------
// compile-time trigonometry: cos/sin(2 pi k / n), exact on the axes
// ---------------------------------------------------------------------------------------
__host__ __device__ constexpr double sin_small(double x) {  // |x| <= pi/4
    const double x2 = x * x;
    return x * (1 - x2 / 6 * (1 - x2 / 20 * (1 - x2 / 42 * (1 - x2 / 72 * (1 - x2 / 110 * (1 - x2 / 156 *
               (1 - x2 / 210 * (1 - x2 / 272))))))));
}
__host__ __device__ constexpr double cos_small(double x) {  // |x| <= pi/4
    const double x2 = x * x;
    return 1 - x2 / 2 * (1 - x2 / 12 * (1 - x2 / 30 * (1 - x2 / 56 * (1 - x2 / 90 * (1 - x2 / 132 *
               (1 - x2 / 182 * (1 - x2 / 240 * (1 - x2 / 306))))))));
}
// cos(2 pi t8 / (8 n)): the angle in eighths of 1/n of a turn, reduced to the first octant in integers
__host__ __device__ constexpr double cos_units(long long t8, long long n) {
    const long long full = 8 * n;
    t8 %= full;
    if (t8 < 0) t8 += full;
    if (t8 > 4 * n) t8 = full - t8;
    bool neg = false;
    if (t8 > 2 * n) { neg = true; t8 = 4 * n - t8; }
    const double two_pi = 6.283185307179586476925286766559;
    const double v = t8 > n ? sin_small(two_pi * (double)(2 * n - t8) / (double)full)
                            : cos_small(two_pi * (double)t8 / (double)full);
    return neg ? -v : v;
}
__host__ __device__ constexpr double cos2pi(long long k, long long n) { return cos_units(8 * k, n); }
__host__ __device__ constexpr double sin2pi(long long k, long long n) { return cos_units(8 * k - 2 * n, n); }

template <int I, int N, typename F>
__device__ __forceinline__ void static_for(F&& f) {
    if constexpr (I < N) {
        f(std::integral_constant<int, I>{});
        static_for<I + 1, N>(f);
    }
}

// a * exp(-2 pi i K / N) with compile-time K, N
template <typename R, int K, int N>
__device__ __forceinline__ Cx<R> mul_w(Cx<R> a) {
    constexpr double c = cos2pi(K, N), s = sin2pi(K, N);
    if constexpr (c == 1.0 && s == 0.0) return a;
    else if constexpr (c == 0.0 && s == 1.0) return mul_mi(a);
    else if constexpr (c == -1.0 && s == 0.0) return mk<R>(-a.re, -a.im);
    else if constexpr (c == 0.0 && s == -1.0) return mul_pi(a);
    else return mk<R>(fma(a.im, R(s), a.re * R(c)), fma(-a.re, R(s), a.im * R(c)));
}

// ---------------------------------------------------------------------------------------
// radix butterflies in registers (forward sign, exp(-2 pi i a q / R)), natural order in and out
// ---------------------------------------------------------------------------------------
constexpr int first_factor(int r) {
    return (r % 4 == 0 && r > 4) ? 4 : (r % 5 == 0 && r > 5) ? 5 : (r % 2 == 0 && r > 2) ? 2
         : (r % 3 == 0 && r > 3) ? 3 : (r % 7 == 0 && r > 7) ? 7 : r;
}

template <typename R, int RAD>
__device__ __forceinline__ void butterfly(Cx<R> (&x)[RAD]) {
    if constexpr (RAD == 2) {
        const Cx<R> a = x[0], b = x[1];
        x[0] = a + b; x[1] = a - b;
    } else if constexpr (RAD == 4) {
        const Cx<R> t0 = x[0] + x[2], t1 = x[0] - x[2], t2 = x[1] + x[3], t3 = mul_mi(x[1] - x[3]);
        x[0] = t0 + t2; x[1] = t1 + t3; x[2] = t0 - t2; x[3] = t1 - t3;
    } else if constexpr (first_factor(RAD) == RAD) {
        // odd prime: pair a with RAD-a;  y_q = A_q - i B_q,  y_{RAD-q} = A_q + i B_q
        constexpr int H = (RAD - 1) / 2;
        Cx<R> t[H + 1], u[H + 1], y[RAD];
        static_for<1, H + 1>([&](auto a_) {
            constexpr int a = a_;
            t[a] = x[a] + x[RAD - a]; u[a] = x[a] - x[RAD - a];
        });
        y[0] = x[0];
        static_for<1, H + 1>([&](auto a_) { constexpr int a = a_; y[0] = y[0] + t[a]; });
        static_for<1, H + 1>([&](auto q_) {
            constexpr int q = q_;
            Cx<R> A = x[0], Bv = mk<R>(R(0), R(0));
            static_for<1, H + 1>([&](auto a_) {
                constexpr int a = a_;
                constexpr double c = cos2pi(a * q, RAD), s = sin2pi(a * q, RAD);
                A.re = fma(R(c), t[a].re, A.re); A.im = fma(R(c), t[a].im, A.im);
                Bv.re = fma(R(s), u[a].re, Bv.re); Bv.im = fma(R(s), u[a].im, Bv.im);
            });
            y[q] = A + mul_mi(Bv);
            y[RAD - q] = A + mul_pi(Bv);
        });
        static_for<0, RAD>([&](auto q_) { constexpr int q = q_; x[q] = y[q]; });
    } else {
        // composite RAD = R1*R2: radix-R1 over stride R2, twiddle exp(-2 pi i a2 q1 / RAD), radix-R2 on
        // each block; slot q1*R2 + q2 then holds bin q1 + R1*q2 - undone by register renaming.
        constexpr int R1 = first_factor(RAD), R2 = RAD / R1;
        static_for<0, R2>([&](auto a2_) {
            constexpr int a2 = a2_;
            Cx<R> t[R1];
            static_for<0, R1>([&](auto a1_) { constexpr int a1 = a1_; t[a1] = x[a2 + R2 * a1]; });
            butterfly<R, R1>(t);
            static_for<0, R1>([&](auto q1_) {
                constexpr int q1 = q1_;
                x[a2 + R2 * q1] = mul_w<R, a2 * q1, RAD>(t[q1]);
            });
        });
        Cx<R> y[RAD];
        static_for<0, R1>([&](auto q1_) {
            constexpr int q1 = q1_;
            Cx<R> t[R2];
            static_for<0, R2>([&](auto a2_) { constexpr int a2 = a2_; t[a2] = x[q1 * R2 + a2]; });
            butterfly<R, R2>(t);
            static_for<0, R2>([&](auto q2_) { constexpr int q2 = q2_; y[q1 + R1 * q2] = t[q2]; });
        });
        static_for<0, RAD>([&](auto q_) { constexpr int q = q_; x[q] = y[q]; });
    }
}

// One decimation-in-frequency pass on every length-Ns block of the N-point array:
//   y_q[j] = w_Ns^{j q} * sum_a x[j + a M] w_R^{a q},  M = Ns/R,  stored in place at j + q M.
// STATIC: N, Ns, M are literals at the call site (this function is inlined), so every stride, bound and division
// below folds to a constant - the planner's common lengths take this route (see fft_inplace).
template <typename R, int T, int RAD, bool STATIC = false>
__device__ __forceinline__ void fft_stage(Cx<R>* __restrict__ sm, const Cx<R>* __restrict__ tw, int N, int Ns,
                                          int M, unsigned magic, int lane_s, int g, int G) {
    const int nb = N / RAD;
    const int tws = (N / Ns) * 2;  // w_Ns = w_L^(2N/Ns)
    const int MT = M * T;
#pragma unroll 1   // one butterfly's registers at a time (the static variants would otherwise unroll this loop)
    for (int u = g; u < nb; u += G) {
        const int blk = M == 1 ? u : STATIC ? u / M : (int)__umulhi((unsigned)u, magic);  // u / M
        const int j = u - blk * M;
        Cx<R>* p = sm + (blk * Ns + j) * T + lane_s;
        Cx<R> x[RAD];
#pragma unroll
        for (int a = 0; a < RAD; ++a) x[a] = p[a * MT];
        butterfly<R, RAD>(x);
        if (M > 1) {
            const Cx<R>* w = tw + j * tws;
#pragma unroll
            for (int q = 1; q < RAD; ++q) x[q] = x[q] * w[(q - 1) * j * tws];
        }
#pragma unroll
        for (int q = 0; q < RAD; ++q) p[q * MT] = x[q];
    }
}

// MAXR = largest register butterfly compiled into the kernel: fp32 kernels take up to radix 25; fp64
// kernels stop at radix 8 so that they stay near 64 registers and four CTAs fit one SM.
template <typename R> struct MaxRadix { static constexpr int value = sizeof(R) == 4 ? 25 : 8; };

// Lengths with a fully static kernel variant (NS template parameter), and their radices - which must be the
// planner's own sequence for that length (tt_api.cu factorise(): largest butterflies first), because the `pos`
// table is built from it; the host only picks a static variant when the plan's radices match.
template <typename R, int NS> struct StaticPlan { static constexpr int r1 = 0, r2 = 0, r3 = 0; };
template <> struct StaticPlan<float, 400> { static constexpr int r1 = 25, r2 = 16, r3 = 1; };
template <> struct StaticPlan<float, 500> { static constexpr int r1 = 25, r2 = 20, r3 = 1; };
template <> struct StaticPlan<float, 256> { static constexpr int r1 = 16, r2 = 16, r3 = 1; };
template <> struct StaticPlan<double, 512> { static constexpr int r1 = 8, r2 = 8, r3 = 8; };
template <> struct StaticPlan<double, 256> { static constexpr int r1 = 8, r2 = 8, r3 = 4; };

template <typename R, int T, int NS = 0>
__device__ __forceinline__ void fft_inplace(Cx<R>* sm, const FftParams& P, int lane_s, int g, int G) {
    constexpr int MAXR = MaxRadix<R>::value;
    const Cx<R>* tw = reinterpret_cast<const Cx<R>*>(P.tw);
    if constexpr (NS != 0 && NS != 500) {   // 500: only the load / post-processing loops are static (registers)
        using SP = StaticPlan<R, NS>;
        constexpr int R1 = SP::r1, R2 = SP::r2, R3 = SP::r3;
        static_assert(R1 * R2 * R3 == NS, "static FFT plan does not match its length");
        __syncthreads();
        fft_stage<R, T, R1, true>(sm, tw, NS, NS, NS / R1, 0u, lane_s, g, G);
        __syncthreads();
        fft_stage<R, T, R2, true>(sm, tw, NS, NS / R1, NS / (R1 * R2), 0u, lane_s, g, G);
        if constexpr (R3 > 1) {
            __syncthreads();
            fft_stage<R, T, R3, true>(sm, tw, NS, R3, 1, 0u, lane_s, g, G);
        }
        __syncthreads();
        return;
    }
    int Ns = P.N;
    for (int st = 0; st < P.n_stages; ++st) {
        __syncthreads();
        const int r = P.radix[st];
        const int M = Ns / r;
        const unsigned mg = P.magic[st];
        switch (r) {
            case 2: fft_stage<R, T, 2>(sm, tw, P.N, Ns, M, mg, lane_s, g, G); break;
            case 3: fft_stage<R, T, 3>(sm, tw, P.N, Ns, M, mg, lane_s, g, G); break;
            case 4: fft_stage<R, T, 4>(sm, tw, P.N, Ns, M, mg, lane_s, g, G); break;
            case 5: fft_stage<R, T, 5>(sm, tw, P.N, Ns, M, mg, lane_s, g, G); break;
            case 7: fft_stage<R, T, 7>(sm, tw, P.N, Ns, M, mg, lane_s, g, G); break;
            case 8: fft_stage<R, T, 8>(sm, tw, P.N, Ns, M, mg, lane_s, g, G); break;
            default:
                if constexpr (MAXR >= 25) {
                    if (r == 16) fft_stage<R, T, 16>(sm, tw, P.N, Ns, M, mg, lane_s, g, G);
                    else if (r == 20) fft_stage<R, T, 20>(sm, tw, P.N, Ns, M, mg, lane_s, g, G);
                    else fft_stage<R, T, 25>(sm, tw, P.N, Ns, M, mg, lane_s, g, G);
                }
                break;
        }
        Ns = M;
    }
    __syncthreads();
}

// The last pass of the inverse kernel (M == 1, Ns == RAD): like fft_stage, but the outputs go straight to global memory
// through io(n, value), n = the bin held by the slot - slot blk*RAD + q holds bin ipos[blk*RAD] + q*(N/RAD), q being the
// most significant digit of the bin index (tt_api.cu build_pos).  No store to shared memory, no barrier, no gather
// through `pos`; and for even RAD the truncation keeps exactly the outputs q < RAD/2, so the other half of the
// butterfly is dead code.  (The mirror image - the forward kernel's first pass reading global memory, with or without
// the zero half of its inputs folded away - was measured slower in both precisions: A1 0.38 -> 0.40 ms at N_t = 400,
// 0.585 -> 0.61 ms at 500, 7.64 -> 7.73 ms for C4's fp64 batch.  The forward path is therefore left exactly as it was.)
template <typename R, int T, int RAD, typename IO>
__device__ __forceinline__ void fft_stage_out(const Cx<R>* __restrict__ sm, int N, int lane_s, int g, int G, const IO& make_io) {
    const int nb = N / RAD;
    const auto io = make_io();
#pragma unroll 1
    for (int u = g; u < nb; u += G) {
        const Cx<R>* p = sm + u * RAD * T + lane_s;
        Cx<R> x[RAD];
#pragma unroll
        for (int a = 0; a < RAD; ++a) x[a] = p[a * T];
        butterfly<R, RAD>(x);
        const int n0 = (int)io.ipos[u * RAD];
#pragma unroll
        for (int q = 0; q < (RAD % 2 == 0 ? RAD / 2 : RAD); ++q) io(n0 + q * nb, x[q]);
    }
}

// fft_inplace for the inverse kernel: every pass but the last as above, the last one through fft_stage_out; there is
// no barrier after it.  N == 1 (no pass): the caller handles it.
template <typename R, int T, int NS, typename IO>
__device__ __forceinline__ void fft_inplace_out(Cx<R>* sm, const FftParams& P, int lane_s, int g, int G, const IO& io) {
    constexpr int MAXR = MaxRadix<R>::value;
    const Cx<R>* tw = reinterpret_cast<const Cx<R>*>(P.tw);
    if constexpr (NS != 0 && NS != 500) {
        using SP = StaticPlan<R, NS>;
        constexpr int R1 = SP::r1, R2 = SP::r2, R3 = SP::r3;
        static_assert(R1 * R2 * R3 == NS, "static FFT plan does not match its length");
        __syncthreads();
        fft_stage<R, T, R1, true>(sm, tw, NS, NS, NS / R1, 0u, lane_s, g, G);
        __syncthreads();
        if constexpr (R3 > 1) {
            fft_stage<R, T, R2, true>(sm, tw, NS, NS / R1, NS / (R1 * R2), 0u, lane_s, g, G);
            __syncthreads();
            fft_stage_out<R, T, R3>(sm, NS, lane_s, g, G, io);
        } else {
            fft_stage_out<R, T, R2>(sm, NS, lane_s, g, G, io);
        }
        return;
    }
    int Ns = P.N;
    for (int st = 0; st + 1 < P.n_stages; ++st) {
        __syncthreads();
        const int r = P.radix[st];
        const int M = Ns / r;
        const unsigned mg = P.magic[st];
        switch (r) {
            case 2: fft_stage<R, T, 2>(sm, tw, P.N, Ns, M, mg, lane_s, g, G); break;
            case 3: fft_stage<R, T, 3>(sm, tw, P.N, Ns, M, mg, lane_s, g, G); break;
            case 4: fft_stage<R, T, 4>(sm, tw, P.N, Ns, M, mg, lane_s, g, G); break;
            case 5: fft_stage<R, T, 5>(sm, tw, P.N, Ns, M, mg, lane_s, g, G); break;
            case 7: fft_stage<R, T, 7>(sm, tw, P.N, Ns, M, mg, lane_s, g, G); break;
            case 8: fft_stage<R, T, 8>(sm, tw, P.N, Ns, M, mg, lane_s, g, G); break;
            default:
                if constexpr (MAXR >= 25) {
                    if (r == 16) fft_stage<R, T, 16>(sm, tw, P.N, Ns, M, mg, lane_s, g, G);
                    else if (r == 20) fft_stage<R, T, 20>(sm, tw, P.N, Ns, M, mg, lane_s, g, G);
                    else fft_stage<R, T, 25>(sm, tw, P.N, Ns, M, mg, lane_s, g, G);
                }
                break;
        }
        Ns = M;
    }
    if (P.n_stages == 0) return;
    __syncthreads();
    switch (Ns) {  // the last radix
        case 2: fft_stage_out<R, T, 2>(sm, P.N, lane_s, g, G, io); break;
        case 3: fft_stage_out<R, T, 3>(sm, P.N, lane_s, g, G, io); break;
        case 4: fft_stage_out<R, T, 4>(sm, P.N, lane_s, g, G, io); break;
        case 5: fft_stage_out<R, T, 5>(sm, P.N, lane_s, g, G, io); break;
        case 7: fft_stage_out<R, T, 7>(sm, P.N, lane_s, g, G, io); break;
        case 8: fft_stage_out<R, T, 8>(sm, P.N, lane_s, g, G, io); break;
        default:
            if constexpr (MAXR >= 25) {
                if (Ns == 16) fft_stage_out<R, T, 16>(sm, P.N, lane_s, g, G, io);
                else if (Ns == 20) fft_stage_out<R, T, 20>(sm, P.N, lane_s, g, G, io);
                else fft_stage_out<R, T, 25>(sm, P.N, lane_s, g, G, io);
            }
            break;
    }
}

// What the inverse kernel's last pass writes: conj(result)_n = z_n * N, x_{2n} = Re z_n, x_{2n+1} = Im z_n, scaled;
// only j < N_t is kept (the truncation)
template <typename Tc>
struct RealStorer {
    Tc* dst;
    long long r_ts;
    const unsigned short* ipos;  // ipos[slot] = bin held by that slot of the in-place DIF output
    int N, dec;
    Tc sc;
    bool live;
    __device__ __forceinline__ void st_real(int j, Tc val) const {  // on a coarser grid only every dec-th time step is kept
        if (dec == 1) dst[(long long)j * r_ts] = val;
        else if ((j + 1) % dec == 0) dst[(long long)((j + 1) / dec - 1) * r_ts] = val;
    }
    __device__ __forceinline__ void operator()(int n, Cx<Tc> v) const {
        if (live && 2 * n < N) {
            st_real(2 * n, v.re * sc);
            if (2 * n + 1 < N) st_real(2 * n + 1, -v.im * sc);
        }
    }
};

}  // namespace tt
