// tt_fft.cu - batched mixed-radix FFTs along time, in shared memory, with the zero-padding,
// the layout change (time-major vectors <-> frequency-major spectra) and the truncation fused
// into the load and the store (steps P0, A1, A3, B1, B3 of DESIGN.md).
//
// One CTA transforms T series at once.  Shared memory holds them as sm[n*T + t] (series index
// fastest), so that the T lanes working on the same butterfly of T different series touch
// consecutive shared-memory words (no bank conflicts) and consecutive global addresses
// (time-major vectors have the space index fastest), and every twiddle factor is uniform over
// those lanes.  The N-point complex FFT is an in-place decimation-in-frequency Cooley-Tukey
// with radices from {2,3,4,5,7}; its digit-reversed output order is undone for free by the
// gather of the following step through the plan's `pos` table.
//
// Real-input trick: the L = 2N-point DFT X of the zero-padded real series x is obtained from
// the N-point DFT Z of z_n = x_{2n} + i x_{2n+1}:
//     X_k = (Z_k + conj Z_{N-k})/2  -  i w^k (Z_k - conj Z_{N-k})/2 ,   w = exp(-2 pi i / L),
// k = 0..N (Z_N := Z_0), and inverted the same way for the real inverse transform.
#include "tt_common.cuh"
#include "tt_internal.h"

namespace tt {

// ---------------------------------------------------------------------------------------
// radix butterflies (forward sign, exp(-2 pi i a q / R))
// ---------------------------------------------------------------------------------------
__host__ __device__ constexpr double tw_cos(int rad, int k) {
    return rad == 3 ? (k == 0 ? 1.0 : -0.5)
         : rad == 5 ? (k == 0 ? 1.0 : (k == 1 || k == 4) ? 0.30901699437494742410 : -0.80901699437494742410)
         : /*7*/      (k == 0 ? 1.0 : (k == 1 || k == 6) ? 0.62348980185873353053
                                    : (k == 2 || k == 5) ? -0.22252093395631440429 : -0.90096886790241912624);
}
__host__ __device__ constexpr double tw_sin(int rad, int k) {  // sin(2 pi k / rad)
    return rad == 3 ? (k == 0 ? 0.0 : k == 1 ? 0.86602540378443864676 : -0.86602540378443864676)
         : rad == 5 ? (k == 0 ? 0.0 : k == 1 ? 0.95105651629515357212 : k == 2 ? 0.58778525229247312917
                                    : k == 3 ? -0.58778525229247312917 : -0.95105651629515357212)
         : /*7*/      (k == 0 ? 0.0 : k == 1 ? 0.78183148246802980871 : k == 2 ? 0.97492791218182360702
                                    : k == 3 ? 0.43388373911755812048 : k == 4 ? -0.43388373911755812048
                                    : k == 5 ? -0.97492791218182360702 : -0.78183148246802980871);
}

template <typename R, int RAD>
__device__ __forceinline__ void butterfly(Cx<R> (&x)[RAD]) {
    if constexpr (RAD == 2) {
        Cx<R> a = x[0], b = x[1];
        x[0] = a + b; x[1] = a - b;
    } else if constexpr (RAD == 4) {
        Cx<R> t0 = x[0] + x[2], t1 = x[0] - x[2], t2 = x[1] + x[3], t3 = mul_mi(x[1] - x[3]);
        x[0] = t0 + t2; x[1] = t1 + t3; x[2] = t0 - t2; x[3] = t1 - t3;
    } else {
        constexpr int H = (RAD - 1) / 2;
        Cx<R> t[H + 1], u[H + 1], y[RAD];
#pragma unroll
        for (int a = 1; a <= H; ++a) { t[a] = x[a] + x[RAD - a]; u[a] = x[a] - x[RAD - a]; }
        y[0] = x[0];
#pragma unroll
        for (int a = 1; a <= H; ++a) y[0] = y[0] + t[a];
#pragma unroll
        for (int q = 1; q <= H; ++q) {
            Cx<R> A = x[0], Bv = mk<R>(R(0), R(0));
#pragma unroll
            for (int a = 1; a <= H; ++a) {
                const R c = R(tw_cos(RAD, (a * q) % RAD)), s = R(tw_sin(RAD, (a * q) % RAD));
                A.re = fma(c, t[a].re, A.re); A.im = fma(c, t[a].im, A.im);
                Bv.re = fma(s, u[a].re, Bv.re); Bv.im = fma(s, u[a].im, Bv.im);
            }
            y[q] = A + mul_mi(Bv);        // A - i B
            y[RAD - q] = A + mul_pi(Bv);  // A + i B
        }
#pragma unroll
        for (int q = 0; q < RAD; ++q) x[q] = y[q];
    }
}

// One decimation-in-frequency stage on every length-Ns block of the N-point array:
//   y_q[j] = w_Ns^{j q} * sum_a x[j + a M] w_R^{a q},  M = Ns/R,  stored in place at j + q M.
template <typename R, int T, int RAD>
__device__ __forceinline__ void fft_stage(Cx<R>* __restrict__ sm, const Cx<R>* __restrict__ tw, int N, int Ns,
                                          int lane_s, int g, int G) {
    const int M = Ns / RAD;
    const int nb = N / RAD;
    const int tws = (N / Ns) * 2;  // w_Ns = w_L^(2N/Ns)
    for (int u = g; u < nb; u += G) {
        const int blk = u / M, j = u - blk * M;
        Cx<R>* p = sm + (size_t)(blk * Ns + j) * T + lane_s;
        Cx<R> x[RAD];
#pragma unroll
        for (int a = 0; a < RAD; ++a) x[a] = p[(size_t)a * M * T];
        butterfly<R, RAD>(x);
        if (M > 1) {
#pragma unroll
            for (int q = 1; q < RAD; ++q) x[q] = x[q] * tw[j * q * tws];
        }
#pragma unroll
        for (int q = 0; q < RAD; ++q) p[(size_t)q * M * T] = x[q];
    }
}

template <typename R, int T>
__device__ __forceinline__ void fft_inplace(Cx<R>* sm, const FftParams& P, int lane_s, int g, int G) {
    const Cx<R>* tw = reinterpret_cast<const Cx<R>*>(P.tw);
    int Ns = P.N;
    for (int st = 0; st < P.n_stages; ++st) {
        __syncthreads();
        const int r = P.radix[st];
        switch (r) {
            case 2: fft_stage<R, T, 2>(sm, tw, P.N, Ns, lane_s, g, G); break;
            case 3: fft_stage<R, T, 3>(sm, tw, P.N, Ns, lane_s, g, G); break;
            case 4: fft_stage<R, T, 4>(sm, tw, P.N, Ns, lane_s, g, G); break;
            case 5: fft_stage<R, T, 5>(sm, tw, P.N, Ns, lane_s, g, G); break;
            default: fft_stage<R, T, 7>(sm, tw, P.N, Ns, lane_s, g, G); break;
        }
        Ns /= r;
    }
    __syncthreads();
}

// ---------------------------------------------------------------------------------------
// forward: zero-pad + real-to-complex FFT + frequency-major store          (P0, A1, B1)
// ---------------------------------------------------------------------------------------
template <typename Tin, typename Tc, typename Tout, int T>
__global__ void fft_r2c_kernel(const Tin* __restrict__ in, Cx<Tout>* __restrict__ out,
                               const __grid_constant__ FftParams P) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Cx<Tc>* sm = reinterpret_cast<Cx<Tc>*>(smem_raw);
    const int lane_s = threadIdx.x % T, g = threadIdx.x / T, G = blockDim.x / T;
    const long long b = (long long)blockIdx.x * T + lane_s;
    const bool live = b < P.B;
    const int N = P.N;
    const Tin* src = in + (long long)blockIdx.y * P.r_ys + b * P.r_bs;

    // z_n = x_{2n} + i x_{2n+1}; x_j = 0 for j >= N_t = N (the zero padding)
    for (int n = g; n < N; n += G) {
        Tc re = Tc(0), im = Tc(0);
        const int j0 = 2 * n;
        if (live && j0 < N) {
            re = Tc(src[(long long)j0 * P.r_ts]);
            if (j0 + 1 < N) im = Tc(src[(long long)(j0 + 1) * P.r_ts]);
        }
        sm[(size_t)n * T + lane_s] = mk<Tc>(re, im);
    }
    fft_inplace<Tc, T>(sm, P, lane_s, g, G);

    const Cx<Tc>* tw = reinterpret_cast<const Cx<Tc>*>(P.tw);
    Cx<Tout>* dst = out + (long long)blockIdx.y * P.c_ys + b * P.c_bs;
    if (b < P.B_store) {
        for (int k = g; k <= N; k += G) {
            const int ka = (k == N) ? 0 : k;
            const int kb = (k == 0 || k == N) ? 0 : N - k;
            const Cx<Tc> Zk = sm[(size_t)P.pos[ka] * T + lane_s];
            const Cx<Tc> Zn = conj(sm[(size_t)P.pos[kb] * T + lane_s]);
            Cx<Tc> E = Zk + Zn, O = mul_mi(Zk - Zn);
            E.re *= Tc(0.5); E.im *= Tc(0.5); O.re *= Tc(0.5); O.im *= Tc(0.5);
            Cx<Tc> X = E + tw[k] * O;
            if (!live) X = mk<Tc>(Tc(0), Tc(0));
            dst[(long long)k * P.c_fs] = mk<Tout>(Tout(X.re), Tout(X.im));
        }
    }
}

// ---------------------------------------------------------------------------------------
// inverse: (sum of partial spectra) + complex-to-real inverse FFT + truncate + scale   (A3, B3)
// ---------------------------------------------------------------------------------------
template <typename Tc, int T>
__global__ void fft_c2r_kernel(const Cx<Tc>* __restrict__ in, Tc* __restrict__ out,
                               const __grid_constant__ FftParams P) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Cx<Tc>* sm = reinterpret_cast<Cx<Tc>*>(smem_raw);
    const int lane_s = threadIdx.x % T, g = threadIdx.x / T, G = blockDim.x / T;
    const long long b = (long long)blockIdx.x * T + lane_s;
    const bool live = b < P.B;
    const int N = P.N;
    const Cx<Tc>* src = in + (long long)blockIdx.y * P.c_ys + b * P.c_bs;

    // X_k, k = 0..N, summed over the partial spectra in fixed order (fp64 accumulator)
    for (int k = g; k <= N; k += G) {
        Cx<Tc> v = mk<Tc>(Tc(0), Tc(0));
        if (live) {
            const Cx<Tc>* q = src + (long long)k * P.c_fs;
            if (P.n_part == 1) {
                v = q[0];
            } else {
                double ar = 0.0, ai = 0.0;
                for (int c = 0; c < P.n_part; ++c) {
                    const Cx<Tc> t = q[(long long)c * P.c_ps];
                    ar += double(t.re); ai += double(t.im);
                }
                v = mk<Tc>(Tc(ar), Tc(ai));
            }
        }
        sm[(size_t)k * T + lane_s] = v;
    }
    __syncthreads();

    // Z_k = (X_k + conj X_{N-k}) + i conj(w^k) (X_k - conj X_{N-k});  store conj(Z_k) so that the
    // forward FFT below yields conj of the inverse transform.  Pairs (k, N-k) are disjoint.
    const Cx<Tc>* tw = reinterpret_cast<const Cx<Tc>*>(P.tw);
    for (int k = g; k <= N / 2; k += G) {
        if (k == 0) {
            const Tc x0 = sm[lane_s].re, xn = sm[(size_t)N * T + lane_s].re;  // DC, Nyquist: real parts only
            sm[lane_s] = mk<Tc>(x0 + xn, -(x0 - xn));
        } else {
            const int kk = N - k;
            const Cx<Tc> Xk = sm[(size_t)k * T + lane_s], Xn = sm[(size_t)kk * T + lane_s];
            const Cx<Tc> Zk = (Xk + conj(Xn)) + mul_pi((Xk - conj(Xn)) * conj(tw[k]));
            if (kk != k) {
                const Cx<Tc> Zkk = (Xn + conj(Xk)) + mul_pi((Xn - conj(Xk)) * conj(tw[kk]));
                sm[(size_t)kk * T + lane_s] = conj(Zkk);
            }
            sm[(size_t)k * T + lane_s] = conj(Zk);
        }
    }
    fft_inplace<Tc, T>(sm, P, lane_s, g, G);

    // conj(result)_n = z_n * N:  x_{2n} = Re z_n, x_{2n+1} = Im z_n; keep j < N_t (truncation)
    if (live) {
        Tc* dst = out + (long long)blockIdx.y * P.r_ys + b * P.r_bs;
        const Tc sc = Tc(P.scale);
        for (int n = g; 2 * n < N; n += G) {
            const Cx<Tc> v = sm[(size_t)P.pos[n] * T + lane_s];
            dst[(long long)(2 * n) * P.r_ts] = v.re * sc;
            if (2 * n + 1 < N) dst[(long long)(2 * n + 1) * P.r_ts] = -v.im * sc;
        }
    }
}

// ---------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------
FftChoice fft_choose(int N, size_t elem) {
    const int Ts[3] = {32, 16, 8};
    FftChoice c{0, 256, 0};
    for (int pass = 0; pass < 2; ++pass) {
        const size_t limit = pass == 0 ? size_t(113) * 1024 : size_t(kMaxSmem);
        for (int i = 0; i < 3; ++i) {
            const size_t bytes = size_t(N + 1) * Ts[i] * elem;
            if (bytes <= limit) { c.T = Ts[i]; c.smem = bytes; return c; }
        }
    }
    return c;
}

template <typename Tin, typename Tc, typename Tout>
static cudaError_t r2c_dispatch(const void* in, void* out, const FftParams& P, int ny, cudaStream_t s) {
    const FftChoice c = fft_choose(P.N, sizeof(Cx<Tc>));
    if (c.T == 0) return cudaErrorInvalidValue;
    const long long nb = (P.B_store > P.B ? P.B_store : P.B);
    dim3 grid((unsigned)((nb + c.T - 1) / c.T), (unsigned)ny);
#define TT_R2C(TT)                                                                                           \
    {                                                                                                        \
        auto k = fft_r2c_kernel<Tin, Tc, Tout, TT>;                                                          \
        cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem);   \
        if (e != cudaSuccess) return e;                                                                      \
        k<<<grid, c.threads, c.smem, s>>>(static_cast<const Tin*>(in), static_cast<Cx<Tout>*>(out), P);      \
    }
    if (c.T == 32) TT_R2C(32) else if (c.T == 16) TT_R2C(16) else TT_R2C(8)
#undef TT_R2C
    return cudaGetLastError();
}

cudaError_t fft_r2c_launch(int tin, int tc, int tout, const void* in, void* out, const FftParams& P, int ny,
                           cudaStream_t s) {
    if (tin == 0 && tc == 0 && tout == 0) return r2c_dispatch<float, float, float>(in, out, P, ny, s);
    if (tin == 0 && tc == 1 && tout == 0) return r2c_dispatch<float, double, float>(in, out, P, ny, s);
    if (tin == 1 && tc == 1 && tout == 1) return r2c_dispatch<double, double, double>(in, out, P, ny, s);
    return cudaErrorInvalidValue;
}

template <typename Tc>
static cudaError_t c2r_dispatch(const void* in, void* out, const FftParams& P, int ny, cudaStream_t s) {
    const FftChoice c = fft_choose(P.N, sizeof(Cx<Tc>));
    if (c.T == 0) return cudaErrorInvalidValue;
    dim3 grid((unsigned)((P.B + c.T - 1) / c.T), (unsigned)ny);
#define TT_C2R(TT)                                                                                           \
    {                                                                                                        \
        auto k = fft_c2r_kernel<Tc, TT>;                                                                     \
        cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem);   \
        if (e != cudaSuccess) return e;                                                                      \
        k<<<grid, c.threads, c.smem, s>>>(static_cast<const Cx<Tc>*>(in), static_cast<Tc*>(out), P);         \
    }
    if (c.T == 32) TT_C2R(32) else if (c.T == 16) TT_C2R(16) else TT_C2R(8)
#undef TT_C2R
    return cudaGetLastError();
}

cudaError_t fft_c2r_launch(int tc, const void* in, void* out, const FftParams& P, int ny, cudaStream_t s) {
    return tc == 0 ? c2r_dispatch<float>(in, out, P, ny, s) : c2r_dispatch<double>(in, out, P, ny, s);
}

}  // namespace tt
