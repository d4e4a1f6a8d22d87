// tt_fft.cu - batched mixed-radix FFTs along time, in shared memory, with the zero-padding,
// the layout change (time-major vectors <-> frequency-major spectra) and the truncation fused
// into the load and the store (steps P0, A1, A3, B1, B3 of DESIGN.md).
//
// One CTA transforms T series at once.  Shared memory holds them as sm[n*T + t] (series index
// fastest), so that the T lanes working on the same butterfly of T different series touch
// consecutive shared-memory words (no bank conflicts) and consecutive global addresses
// (time-major vectors have the space index fastest), and every twiddle factor is uniform over
// those lanes.  The N-point complex FFT is an in-place decimation-in-frequency Cooley-Tukey.
// A pass is a radix-R butterfly done entirely in registers, R from {2,3,4,5,7} or a composite
// {8,16,20,25} built from those at compile time (so N = 400 = 16*25 is two passes over shared
// memory, 512 = 16*8*4 three); the digit-reversed output order of the passes is undone for
// free by the gather of the following step through the plan's `pos` table.
//
// Real-input trick: the L = 2N-point DFT X of the zero-padded real series x is obtained from
// the N-point DFT Z of z_n = x_{2n} + i x_{2n+1}:
//     X_k = (Z_k + conj Z_{N-k})/2  -  i w^k (Z_k - conj Z_{N-k})/2 ,   w = exp(-2 pi i / L),
// k = 0..N (Z_N := Z_0), and inverted the same way for the real inverse transform.
#include "tt_fft_device.cuh"

namespace tt {

double debug_cos2pi(long long k, long long n) { return cos2pi(k, n); }
double debug_sin2pi(long long k, long long n) { return sin2pi(k, n); }

// ---------------------------------------------------------------------------------------
// forward: zero-pad + real-to-complex FFT + frequency-major store          (P0, A1, B1)
// ---------------------------------------------------------------------------------------
// The static 400 variant is held to 64 registers so that FOUR CTAs share an SM (its 51 KB tiles allow it): the phases of a
// CTA are serial, resident neighbours are what overlaps loads with butterflies - A1 0.445 -> 0.380 ms, B3 0.551 -> 0.479 ms.
template <typename Tin, typename Tc, typename Tout, int T, int NT, int NS = 0>
__global__ void __launch_bounds__(NT, NS == 400 ? 4 : (NS == 500 || NT == 320) ? 3 : 0)
fft_r2c_kernel(const Tin* __restrict__ in, Cx<Tout>* __restrict__ out, const __grid_constant__ FftParams P) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Cx<Tc>* sm = reinterpret_cast<Cx<Tc>*>(smem_raw);
    constexpr int G = NT / T;
    const int lane_s = threadIdx.x % T, g = threadIdx.x / T;
    const long long b = (long long)blockIdx.x * T + lane_s;
    const bool live = b < P.B;
    const int N = NS ? NS : P.N;
    const Tin* src = in + (long long)blockIdx.y * P.r_ys + b * P.r_bs;
    const int dec = P.dec;
    auto ld_real = [&](int j) -> Tin {   // time step j of the series; on a coarser grid only every dec-th step exists
        if (dec == 1) return src[(long long)j * P.r_ts];
        return ((j + 1) % dec == 0) ? src[(long long)((j + 1) / dec - 1) * P.r_ts] : Tin(0);
    };

    // z_n = x_{2n} + i x_{2n+1}; x_j = 0 for j >= N_t = N (the zero padding).  The global loads are
    // issued in batches of 2*UB independent requests per thread before any of them is consumed.
    constexpr int UB = 8;
    const int nh = (N + 1) / 2;  // slots n >= nh are pure padding
    for (int n0 = g; n0 < nh; n0 += G * UB) {
        Tin v0[UB], v1[UB];
#pragma unroll
        for (int u = 0; u < UB; ++u) {
            const int n = n0 + u * G;
            v0[u] = Tin(0); v1[u] = Tin(0);
            if (live && n < nh) {
                v0[u] = ld_real(2 * n);
                if (2 * n + 1 < N) v1[u] = ld_real(2 * n + 1);
            }
        }
#pragma unroll
        for (int u = 0; u < UB; ++u) {
            const int n = n0 + u * G;
            if (n < nh) sm[n * T + lane_s] = mk<Tc>(Tc(v0[u]), Tc(v1[u]));
        }
    }
    for (int n = nh + g; n < N; n += G) sm[n * T + lane_s] = mk<Tc>(Tc(0), Tc(0));
    fft_inplace<Tc, T, NS>(sm, P, lane_s, g, G);

    const Cx<Tc>* tw = reinterpret_cast<const Cx<Tc>*>(P.tw);
    Cx<Tout>* dst = out + (long long)blockIdx.y * P.c_ys + b * P.c_bs;
    if (b < P.B_store) {
        // bins k and N-k share their inputs:  X_k = E + w^k O,  X_{N-k} = conj(E - w^k O)
        // slot of bin k: arithmetic for the static fp64 variants (digits of k in the plan's radices: A1 0.47 -> 0.415 ms at
        // N_t = 256), the `pos` table otherwise (the fp32 variants were measured 3 % slower with the arithmetic)
        auto slot = [&](int k) -> int {
            if constexpr (NS != 0 && sizeof(Tc) == 8) {
                using SP = StaticPlan<Tc, NS>;
                constexpr int R1 = SP::r1, R2 = SP::r2, R3 = SP::r3;
                const int q1 = k % R1, r = k / R1;
                if constexpr (R3 > 1) return q1 * (NS / R1) + (r % R2) * R3 + r / R2;
                else return q1 * R2 + r;
            } else {
                return (int)P.pos[k];
            }
        };
        for (int k = g; k <= N / 2; k += G) {
            const int kk = N - k;
            const Cx<Tc> Zk = sm[slot(k) * T + lane_s];
            const Cx<Tc> Zn = conj(sm[slot(k == 0 ? 0 : kk) * T + lane_s]);
            Cx<Tc> E = Zk + Zn, O = mul_mi(Zk - Zn);
            E.re *= Tc(0.5); E.im *= Tc(0.5); O.re *= Tc(0.5); O.im *= Tc(0.5);
            const Cx<Tc> wO = tw[k] * O;
            Cx<Tc> Xa = E + wO, Xb = conj(E - wO);
            if (!live) { Xa = mk<Tc>(Tc(0), Tc(0)); Xb = Xa; }
            dst[(long long)k * P.c_fs] = mk<Tout>(Tout(Xa.re), Tout(Xa.im));
            if (kk != k) dst[(long long)kk * P.c_fs] = mk<Tout>(Tout(Xb.re), Tout(Xb.im));
        }
    }
}

// ---------------------------------------------------------------------------------------
// inverse: complex-to-real inverse FFT + truncate + scale                               (A3, B3)
// ---------------------------------------------------------------------------------------
// One tile of T series (tile index `tile`, grid row `by`): shared by the one-CTA-per-tile kernel and the persistent consumer.
// STREAMED: the input was parked in the L2 by the kernel that produced it (tt_gemv.cu, L2R) and is read exactly once here:
// it is loaded past L1 and its lines are dropped from the L2 afterwards without a write-back (whole 128-byte lines per tile).
template <typename Tc, int T, int NT, int NS, bool STREAMED = false>
__device__ __forceinline__ void c2r_tile(const Cx<Tc>* __restrict__ in, Tc* __restrict__ out, const FftParams& P, long long tile, int by) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Cx<Tc>* sm = reinterpret_cast<Cx<Tc>*>(smem_raw);
    constexpr int G = NT / T;
    const int lane_s = threadIdx.x % T, g = threadIdx.x / T;
    const long long b = tile * T + lane_s;
    const bool live = b < P.B;
    const int N = NS ? NS : P.N;
    const Cx<Tc>* src = in + (long long)by * P.c_ys + b * P.c_bs;

    // Z_k = (X_k + conj X_{N-k}) + i conj(w^k) (X_k - conj X_{N-k});  store conj(Z_k) so that the
    // forward FFT below yields conj of the inverse transform.  Pairs (k, N-k) are disjoint; both members are read
    // from global memory by the thread that needs them, in batches of 2*UB independent requests.
    const Cx<Tc>* tw = reinterpret_cast<const Cx<Tc>*>(P.tw);
    constexpr int UB = 4;
    const int nh = N / 2;
    for (int k0 = g; k0 <= nh; k0 += G * UB) {
        Cx<Tc> va[UB], vb[UB];
#pragma unroll
        for (int u = 0; u < UB; ++u) {
            const int k = k0 + u * G;
            va[u] = mk<Tc>(Tc(0), Tc(0)); vb[u] = va[u];
            if (live && k <= nh) {
                if constexpr (STREAMED) {
                    va[u] = ld_cg(src + (long long)k * P.c_fs);
                    vb[u] = ld_cg(src + (long long)(N - k) * P.c_fs);
                } else {
                    va[u] = src[(long long)k * P.c_fs];
                    vb[u] = src[(long long)(N - k) * P.c_fs];
                }
            }
        }
#pragma unroll
        for (int u = 0; u < UB; ++u) {
            const int k = k0 + u * G;
            if (k > nh) continue;
            if (k == 0) {
                const Tc x0 = va[u].re, xn = vb[u].re;  // DC, Nyquist: real parts only
                sm[lane_s] = mk<Tc>(x0 + xn, -(x0 - xn));
            } else {
                const int kk = N - k;
                const Cx<Tc> Xk = va[u], Xn = vb[u];
                const Cx<Tc> Zk = (Xk + conj(Xn)) + mul_pi((Xk - conj(Xn)) * conj(tw[k]));
                if (kk != k) {
                    const Cx<Tc> Zkk = (Xn + conj(Xk)) + mul_pi((Xn - conj(Xk)) * conj(tw[kk]));
                    sm[kk * T + lane_s] = conj(Zkk);
                }
                sm[k * T + lane_s] = conj(Zk);
            }
        }
    }
    if constexpr (STREAMED) {
        constexpr int LINES = (int)(T * sizeof(Cx<Tc>) / 128);   // whole lines per frequency row of the tile (the host checks)
        if (P.discard_in) {
            __syncthreads();   // every load of the tile has returned (its value went to shared memory)
            const char* base = reinterpret_cast<const char*>(in + (long long)by * P.c_ys + tile * T * P.c_bs);
            for (int i = threadIdx.x; i < (N + 1) * LINES; i += NT)
                l2_discard_line(base + (long long)(i / LINES) * P.c_fs * (long long)sizeof(Cx<Tc>) + (i % LINES) * 128);
        }
    }
    // built where it is used (after the passes over shared memory), so that its fields are not live across them
    auto stz = [&]() {
        return RealStorer<Tc>{out + (long long)by * P.r_ys + b * P.r_bs, P.r_ts, P.pos + N, N, P.dec, Tc(P.scale), live};
    };
    if (N == 1) {  // no pass
        __syncthreads();
        if (g == 0) stz()(0, sm[lane_s]);
    }
    fft_inplace_out<Tc, T, NS>(sm, P, lane_s, g, G, stz);
}

template <typename Tc, int T, int NT, int NS = 0>
__global__ void __launch_bounds__(NT, NS == 400 ? 4 : (NS == 500 || NT == 320 || (NS == 0 && NT == 256 && sizeof(Tc) == 4)) ? 3 : 0)
fft_c2r_kernel(const Cx<Tc>* __restrict__ in, Tc* __restrict__ out, const __grid_constant__ FftParams P) {
    if (P.skip && P.skip[blockIdx.x]) return;   // done by the consumer kernel while B2 was running
    c2r_tile<Tc, T, NT, NS>(in, out, P, (long long)blockIdx.x, (int)blockIdx.y);
}

// B3 as the CONSUMER of a running B2 (tt_api.cu run_rmatvec, L2R): a few persistent CTAs take the tiles of T series in
// ascending order from a ticket, wait until all N + 1 frequencies of the tile's parameters have been stored by B2 (one
// counter per B2 tile of `ptile` parameters, incremented by every B2 CTA after its store), transform the tile, store the
// truncated real series and flag the tile as done.  The spectrum is read where B2 parked it, in the L2, and dropped there.
// The consumer is an ACCELERATOR, not a dependency: a CTA that waits 50 ms for a counter (B2 is not running beside it - a
// profiler or debugger that serialises kernels, a GPU shared with other work) gives up, and the regular B3 launch that
// follows B2 on the caller's stream transforms every tile that carries no done flag.
//   sync[0] = ticket, sync[2 + i] = counter of B2 tile i;  done[t] = 1: tile t of T series is finished
template <typename Tc, int T, int NT, int NS = 0>
__global__ void __launch_bounds__(NT, 3)   // <= 80 registers: three or four of B2's CTAs share the SM with one of these
fft_c2r_consumer_kernel(const Cx<Tc>* __restrict__ in, Tc* __restrict__ out, const __grid_constant__ FftParams P,
                        unsigned* sync, unsigned char* done, long long n_tiles, int ptile, unsigned n_f) {
    __shared__ long long s_tile;
    for (;;) {
        __syncthreads();   // the previous tile's last pass has read shared memory
        if (threadIdx.x == 0) {
            // Once B2's LAST tile is complete B2 is (all but) over and the whole GPU is free: the few tiles that are left are
            // quicker in the clean-up launch (one CTA per tile on every SM) than in these few CTAs - take no more.
            unsigned last;
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(last) : "l"(sync + 2 + ((n_tiles - 1) * T) / ptile) : "memory");
            long long t = last >= n_f ? n_tiles : (long long)atomicAdd(sync, 1u);
            if (t < n_tiles) {
                const unsigned* cnt = sync + 2 + (t * T) / ptile;
                unsigned long long t0, t1;
                asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
                unsigned v;
                for (;;) {
                    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(cnt) : "memory");
                    if (v >= n_f) break;
                    __nanosleep(256);
                    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
                    if (t1 - t0 > 50000000ULL) { t = n_tiles; break; }   // 50 ms: the producer is not running beside us
                }
                if (t < n_tiles) done[t] = 1;   // taken and never abandoned from here on: the clean-up launch (after this kernel) skips it
            }
            s_tile = t;
        }
        __syncthreads();
        const long long tile = s_tile;
        if (tile >= n_tiles) break;
        c2r_tile<Tc, T, NT, NS, true>(in, out, P, tile, 0);
    }
}

// ---------------------------------------------------------------------------------------
// A3 helper: dhat[w][s] = sum_c partial[w][c][s], fixed order, fp64 accumulator
// ---------------------------------------------------------------------------------------
template <typename R>
__global__ void __launch_bounds__(256)
reduce_partials_kernel(const Cx<R>* __restrict__ partial, Cx<R>* __restrict__ dhat, int n_f, int n_chunks, int N_d) {
    const int w = blockIdx.y;
    const int s = blockIdx.x * 256 + threadIdx.x;
    if (s >= N_d) return;
    const Cx<R>* q = partial + (long long)w * n_chunks * N_d + s;
    double ar = 0.0, ai = 0.0;
    int c = 0;
    for (; c + 8 <= n_chunks; c += 8) {
        Cx<R> t[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) t[u] = q[(long long)(c + u) * N_d];
#pragma unroll
        for (int u = 0; u < 8; ++u) { ar += double(t[u].re); ai += double(t[u].im); }
    }
    for (; c < n_chunks; ++c) {
        const Cx<R> t = q[(long long)c * N_d];
        ar += double(t.re); ai += double(t.im);
    }
    dhat[(long long)w * N_d + s] = mk<R>(R(ar), R(ai));
}

cudaError_t reduce_partials_launch(int dt, const void* partial, void* dhat, int n_f, int n_chunks, int N_d,
                                   cudaStream_t s) {
    dim3 grid((unsigned)((N_d + 255) / 256), (unsigned)n_f);
    if (dt == 0)
        reduce_partials_kernel<float><<<grid, 256, 0, s>>>(static_cast<const c64*>(partial), static_cast<c64*>(dhat),
                                                           n_f, n_chunks, N_d);
    else
        reduce_partials_kernel<double><<<grid, 256, 0, s>>>(static_cast<const c128*>(partial),
                                                            static_cast<c128*>(dhat), n_f, n_chunks, N_d);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------
static int g_force_T = 0, g_force_NT = 0, g_no_static = 0;
void fft_debug_no_static(int v) { g_no_static = v; }
void fft_debug_force_T(int T) { g_force_T = T; }
void fft_debug_force_threads(int NT) { g_force_NT = NT; }

FftChoice fft_choose(int N, size_t elem) {
    // Measured on B200 (C2, C3, C5 shapes, both precisions): 256 threads and T = 16 series per CTA win as
    // long as >= 3 CTAs fit one SM's shared memory; the phases of a CTA (global load, passes, store) are
    // serial, so several resident CTAs are what overlaps HBM traffic with the butterflies.
    FftChoice c{0, 256, 0};
    auto bytes = [&](int T) { return size_t(N + 1) * T * elem; };
    if (g_force_T) {
        if (bytes(g_force_T) <= size_t(kMaxSmem)) { c.T = g_force_T; c.smem = bytes(g_force_T); return c; }
    }
    const int order[3] = {16, 8, 32};
    const size_t limits[3] = {size_t(76) * 1024, size_t(113) * 1024, size_t(kMaxSmem)};
    for (int pass = 0; pass < 3; ++pass)
        for (int i = 0; i < (pass == 0 ? 3 : 2); ++i)
            if (bytes(order[i]) <= limits[pass]) { c.T = order[i]; c.smem = bytes(order[i]); return c; }
    return c;
}

// The static variant for this plan, or 0: T = 16 / 256 threads only (the planner's choice for these lengths), and the
// plan's radices must be the ones compiled in.
template <typename Tc>
static int static_length(const FftParams& P, const FftChoice& c, int nt, bool inverse) {
    if (g_no_static > 0 || nt != 256) return 0;
    // fp64, N_t = 512 (C4's batched transforms run with T = 8): static kernels 6 % faster (forward: with the arithmetic slots)
    if (sizeof(Tc) == 8 && c.T == 8) return (P.N == 512 && P.n_stages == 3 && P.radix[0] == 8 && P.radix[1] == 8 && P.radix[2] == 8) ? 512 : 0;
    if (c.T != 16) return 0;
    auto is = [&](int n, int r1, int r2, int r3) {
        return P.N == n && P.n_stages == (r3 > 1 ? 3 : 2) && P.radix[0] == r1 && P.radix[1] == r2 &&
               (r3 == 1 || P.radix[2] == r3);
    };
    // 500 = 25 x 20: fully static passes need ~130 registers (slower); only the load / post-processing loops are static
    // there, and only in the forward kernel (A1 0.63 -> 0.585 ms; the inverse kernel spills and was measured slower)
    if (sizeof(Tc) == 4)
        return is(400, 25, 16, 1) ? 400 : (!inverse && is(500, 25, 20, 1)) ? 500 : is(256, 16, 16, 1) ? 256 : 0;
    return is(512, 8, 8, 8) ? 512 : is(256, 8, 8, 4) ? 256 : 0;
}

template <typename Tin, typename Tc, typename Tout>
static cudaError_t r2c_dispatch(const void* in, void* out, const FftParams& P, int ny, cudaStream_t s) {
    const FftChoice c = fft_choose(P.N, sizeof(Cx<Tc>));
    if (c.T == 0) return cudaErrorInvalidValue;
    const int nt = g_force_NT ? g_force_NT : 256;
    const long long nb = (P.B_store > P.B ? P.B_store : P.B);
    dim3 grid((unsigned)((nb + c.T - 1) / c.T), (unsigned)ny);
#define TT_R2C(TT, NT, ...)                                                                                  \
    {                                                                                                        \
        auto k = fft_r2c_kernel<Tin, Tc, Tout, TT, NT, ##__VA_ARGS__>;                                                    \
        cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem);   \
        if (e != cudaSuccess) return e;                                                                      \
        k<<<grid, NT, c.smem, s>>>(static_cast<const Tin*>(in), static_cast<Cx<Tout>*>(out), P);             \
    }
    const int ns = static_length<Tc>(P, c, nt, false);
    if (ns) {
        if constexpr (sizeof(Tc) == 4) { if (ns == 400) TT_R2C(16, 256, 400) else if (ns == 500) TT_R2C(16, 256, 500) else TT_R2C(16, 256, 256) }
        else                           { if (ns == 512 && c.T == 8) TT_R2C(8, 256, 512) else if (ns == 512) TT_R2C(16, 256, 512) else TT_R2C(16, 256, 256) }
    }
    else if (nt == 512) { if (c.T == 32) TT_R2C(32, 512) else if (c.T == 16) TT_R2C(16, 512) else TT_R2C(8, 512) }
    else                { if (c.T == 32) TT_R2C(32, 256) else if (c.T == 16) TT_R2C(16, 256) else TT_R2C(8, 256) }
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
    // N_t = 500 = 25 x 20: 320 butterflies per pass-1 round of 16 series - ten warps do it in one round and three such
    // CTAs at 64 registers share an SM: B3 0.76 -> 0.69 ms (the forward kernel was measured slower that way)
    const int nt = g_force_NT ? g_force_NT : (sizeof(Tc) == 4 && P.N == 500 && c.T == 16) ? 320 : 256;
    dim3 grid((unsigned)((P.B + c.T - 1) / c.T), (unsigned)ny);
#define TT_C2R(TT, NT, ...)                                                                                  \
    {                                                                                                        \
        auto k = fft_c2r_kernel<Tc, TT, NT, ##__VA_ARGS__>;                                                               \
        cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem);   \
        if (e != cudaSuccess) return e;                                                                      \
        k<<<grid, NT, c.smem, s>>>(static_cast<const Cx<Tc>*>(in), static_cast<Tc*>(out), P);                \
    }
    const int ns = static_length<Tc>(P, c, nt, true);
    if (ns) {
        if constexpr (sizeof(Tc) == 4) { if (ns == 400) TT_C2R(16, 256, 400) else if (ns == 500) TT_C2R(16, 256, 500) else TT_C2R(16, 256, 256) }
        else                           { if (ns == 512 && c.T == 8) TT_C2R(8, 256, 512) else if (ns == 512) TT_C2R(16, 256, 512) else TT_C2R(16, 256, 256) }
    }
    else if (nt == 320 && c.T == 16) { if constexpr (sizeof(Tc) == 4) TT_C2R(16, 320) }
    else if (nt == 512) { if (c.T == 32) TT_C2R(32, 512) else if (c.T == 16) TT_C2R(16, 512) else TT_C2R(8, 512) }
    else                { if (c.T == 32) TT_C2R(32, 256) else if (c.T == 16) TT_C2R(16, 256) else TT_C2R(8, 256) }
#undef TT_C2R
    return cudaGetLastError();
}

// The persistent consumer (see fft_c2r_consumer_kernel): the plan's usual variant for this length, n_ctas CTAs.
template <typename Tc>
static cudaError_t c2r_consumer_dispatch(const void* in, void* out, const FftParams& P, unsigned* sync, unsigned char* done,
                                         int ptile, int n_ctas, cudaStream_t s) {
    const FftChoice c = fft_choose(P.N, sizeof(Cx<Tc>));
    if (c.T == 0 || (c.T * sizeof(Cx<Tc>)) % 128 != 0 || ptile % c.T != 0 || P.c_bs != 1) return cudaErrorInvalidValue;
    const long long n_tiles = (P.B + c.T - 1) / c.T;
    const unsigned n_f = (unsigned)P.N + 1u;
#define TT_C2RC(TT, ...)                                                                                      \
    {                                                                                                        \
        auto k = fft_c2r_consumer_kernel<Tc, TT, 256, ##__VA_ARGS__>;                                         \
        cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.smem);   \
        if (e != cudaSuccess) return e;                                                                      \
        k<<<n_ctas, 256, c.smem, s>>>(static_cast<const Cx<Tc>*>(in), static_cast<Tc*>(out), P, sync, done, n_tiles, ptile, n_f); \
    }
    const int ns = static_length<Tc>(P, c, 256, true);
    if (ns) {
        if constexpr (sizeof(Tc) == 4) { if (ns == 400) TT_C2RC(16, 400) else if (ns == 500) TT_C2RC(16, 500) else TT_C2RC(16, 256) }
        else                           { if (ns == 512 && c.T == 8) TT_C2RC(8, 512) else if (ns == 512) TT_C2RC(16, 512) else TT_C2RC(16, 256) }
    }
    else { if (c.T == 32) TT_C2RC(32) else if (c.T == 16) TT_C2RC(16) else TT_C2RC(8) }
#undef TT_C2RC
    return cudaGetLastError();
}

bool fft_c2r_consumer_ok(int tc, int N, int ptile) {
    const size_t cs = tc == 0 ? sizeof(c64) : sizeof(c128);
    const FftChoice c = fft_choose(N, cs);
    return c.T != 0 && (c.T * cs) % 128 == 0 && ptile % c.T == 0;
}

cudaError_t fft_c2r_consumer_launch(int tc, const void* in, void* out, const FftParams& P, unsigned* sync, unsigned char* done,
                                    int ptile, int n_ctas, cudaStream_t s) {
    return tc == 0 ? c2r_consumer_dispatch<float>(in, out, P, sync, done, ptile, n_ctas, s)
                   : c2r_consumer_dispatch<double>(in, out, P, sync, done, ptile, n_ctas, s);
}

cudaError_t fft_c2r_launch(int tc, const void* in, void* out, const FftParams& P, int ny, cudaStream_t s) {
    return tc == 0 ? c2r_dispatch<float>(in, out, P, ny, s) : c2r_dispatch<double>(in, out, P, ny, s);
}

}  // namespace tt
