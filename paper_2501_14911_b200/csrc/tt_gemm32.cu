// tt_gemm32.cu - k right-hand sides at once for TT_F32 plans: the per-frequency products as complex64 GEMMs
//     forward   Dhat_w [N_d x k] = Fhat_w   [N_d x N_m] * Xhat_w [N_m x k]
//     adjoint   Xhat_w [N_m x k] = Fhat_w^H [N_m x N_d] * Dhat_w [N_d x k]
// (step D of DESIGN.md for fp32; the many-matvec workloads of PAPER.md:296, 407, 421-423 - K assembly pushes
// N_d N_t unit vectors through G* and F).  With k = 32 columns every Fhat byte feeds 32 flop, far above the
// ~10 flop/B at which the FP32 FMA pipe saturates, so these are compute-bound register-tiled FMA GEMMs.  They are the
// path for the shapes the tcgen05 3xTF32 kernels (tt_gemm32_umma.cu) do not take: k not a multiple of 16, and the
// adjoint with N_d > 128.
// Operands are staged in shared memory with a 2-stage cp.async pipeline; all sums have a fixed order.
#include "tt_common.cuh"
#include "tt_internal.h"

namespace tt {

namespace {

int g_fwd_variant = 0;   // tuning hook: 0 = planner's choice


// Measured and rejected: packed fma.rn.f32x2 (SASS FFMA2) for the complex MACs - the register-pair shuffles
// (a.re, a.re), (-a.im, a.im), (b.im, b.re) cost one MOV per FFMA2 and the kernels ran 1.2-1.3x slower on B200.

// The 4 columns of column group tx: {2tx, 2tx+1} and {2 NCG + 2tx, 2 NCG + 2tx + 1}, so that the 8 (or 4) lanes of a
// quarter-warp read 16-byte pieces of the Xhat / Dhat tile that are CONTIGUOUS (two pieces per lane at stride 32 B cost
// twice the shared-memory wavefronts: ncu, 8 instead of 4 per LDS.128).
template <int NCG>
__device__ __forceinline__ int thread_col(int tx, int j) { return (j < 2 ? 0 : 2 * NCG) + 2 * tx + (j & 1); }

constexpr int KP = 32;        // forward: parameters per pipeline stage
constexpr int AP = KP + 2;    // A-tile pitch in complex elements (272 B: 16-byte aligned rows, skewed banks)
constexpr int NC = 32;        // columns per launch: NCG = 8 column groups of 4 (NCG = 4 when only <= 16 are left)

// ---------------------------------------------------------------------------------------
// forward: partial[((w*nsplit + c)*N_d + s)*k + r0 + r] = sum_{p in split c} Fhat_w[s,p] Xhat_w[p, r0 + r]
// grid (nsplit, n_f, ceil(N_d / (TY TS))), 8 TY threads = TY sensor rows x 8 column groups; a thread owns TS
// sensors (ty, ty + TY, ...) x 4 columns (thread_col).  Shared-memory bandwidth bounds this kernel (every thread re-reads its
// 4 columns of the Xhat tile per parameter), so the sensor tile per thread is made as tall as N_d allows.
// ---------------------------------------------------------------------------------------
template <int TS, int TY, int NCG>
__global__ void __launch_bounds__(NCG * TY)
gemm32_fwd_kernel(const c64* __restrict__ Fhat, const c64* __restrict__ Xhat, c64* __restrict__ partial,
                  const GemmGeom g, const int r0, const int kk) {
    constexpr int ROWS = TY * TS, NT = NCG * TY, NCW = 4 * NCG;   // NCW = columns of the Xhat tile
    extern __shared__ __align__(16) unsigned char smem_raw[];
    c64* As = reinterpret_cast<c64*>(smem_raw);          // [2][ROWS][AP]
    c64* Bs = As + 2 * ROWS * AP;                         // [2][KP][NCW]

    const int tid = threadIdx.x, tx = tid % NCG, ty = tid / NCG;
    const int w = blockIdx.y, c = blockIdx.x, s0 = blockIdx.z * ROWS;
    const long long p_lo = (long long)c * g.p_per_split;
    long long p_hi = p_lo + g.p_per_split;
    if (p_hi > g.N_m) p_hi = g.N_m;
    const int n_it = p_hi > p_lo ? (int)((p_hi - p_lo + KP - 1) / KP) : 0;
    const c64* Abase = Fhat + ((long long)w * g.N_d + s0) * g.ldp;
    const c64* Bbase = Xhat + (long long)w * g.ldx + r0;

    auto load_stage = [&](int st, int it) {
        const long long p0 = p_lo + (long long)it * KP;
        c64* a = As + st * ROWS * AP;
#pragma unroll
        for (int i = 0; i < (ROWS * KP / 2) / NT; ++i) {        // 16-byte chunks = 2 complex64 (pad of Fhat rows is zero)
            const int e = i * NT + tid, row = e / (KP / 2), col = (e % (KP / 2)) * 2;
            const bool ok = (s0 + row < g.N_d) && (p0 + col < p_hi);
            cp_async16(a + row * AP + col, ok ? Abase + (long long)row * g.ldp + p0 + col : Abase, ok);
        }
        c64* b = Bs + st * KP * NCW;
#pragma unroll
        for (int i = 0; i < (KP * NCW) / NT; ++i) {             // 8-byte chunks: rows of Xhat_w need not be 16-byte aligned
            const int e = i * NT + tid, row = e / NCW, col = e % NCW;
            const bool ok = (p0 + row < p_hi) && (col < kk);
            cp_async8(b + row * NCW + col, ok ? Bbase + (p0 + row) * (long long)g.k + col : Bbase, ok);
        }
    };

    c64 acc[TS][4];
#pragma unroll
    for (int i = 0; i < TS; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = mk<float>(0.f, 0.f);

    if (n_it > 0) load_stage(0, 0);
    cp_async_commit();
    for (int it = 0; it < n_it; ++it) {
        cp_async_wait_all();
        __syncthreads();
        if (it + 1 < n_it) load_stage((it + 1) & 1, it + 1);
        cp_async_commit();
        const c64* a = As + (it & 1) * ROWS * AP + ty * AP;
        const float4* b = reinterpret_cast<const float4*>(Bs + (it & 1) * KP * NCW) + tx;
#pragma unroll 8
        for (int p = 0; p < KP; ++p) {
            const float4 b01 = b[p * (NCW / 2)], b23 = b[p * (NCW / 2) + NCG];   // 8 lanes x 16 B contiguous: no bank conflict
            const c64 bv[4] = {mk<float>(b01.x, b01.y), mk<float>(b01.z, b01.w), mk<float>(b23.x, b23.y),
                               mk<float>(b23.z, b23.w)};
#pragma unroll
            for (int i = 0; i < TS; ++i) {
                const c64 av = a[i * TY * AP + p];
#pragma unroll
                for (int j = 0; j < 4; ++j) cmac(acc[i][j], av, bv[j]);
            }
        }
    }
#pragma unroll
    for (int i = 0; i < TS; ++i) {
        const int s = s0 + ty + TY * i;
        if (s >= g.N_d) continue;
        c64* dst = partial + (((long long)w * g.split + c) * g.N_d + s) * g.k + r0;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int col = thread_col<NCG>(tx, j);
            if (col < kk) dst[col] = acc[i][j];
        }
    }
}

// ---------------------------------------------------------------------------------------
// adjoint: Xout_w[p, r0 + r] = sum_s conj(Fhat_w[s,p]) Dhat_w[s, r0 + r]
// grid (ceil(ldp/256), n_f), 256 threads = 32 parameter groups x 8 column groups; a thread owns
// 8 consecutive parameters x 4 columns.  Dhat_w (N_d x 32) sits in shared memory for the whole CTA,
// Fhat_w rows (2 KB contiguous per sensor) go through a 2-stage cp.async pipeline, KS sensors per stage.
// ---------------------------------------------------------------------------------------
constexpr int KS = 8;

template <int NCG>
__global__ void __launch_bounds__(256, 2)
gemm32_adj_kernel(const c64* __restrict__ Fhat, const c64* __restrict__ Dhat, c64* __restrict__ Xout,
                  const GemmGeom g, const int r0, const int kk) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int PT = 8 * (256 / NCG), NCW = 4 * NCG;    // parameters per CTA, columns of the Dhat tile
    c64* As = reinterpret_cast<c64*>(smem_raw);          // [2][KS][PT]
    c64* Ds = As + 2 * KS * PT;                           // [N_d][NCW]

    const int tid = threadIdx.x, tx = tid % NCG, ty = tid / NCG;
    const int w = blockIdx.y;
    const long long p0 = (long long)blockIdx.x * PT;
    const c64* Abase = Fhat + (long long)w * g.N_d * g.ldp + p0;
    const c64* Dbase = Dhat + (long long)w * g.N_d * g.k + r0;
    const int n_it = (g.N_d + KS - 1) / KS;

    for (int e = tid; e < g.N_d * NCW; e += 256) {
        const int s = e / NCW, col = e % NCW;
        Ds[e] = col < kk ? Dbase[(long long)s * g.k + col] : mk<float>(0.f, 0.f);
    }
    auto load_stage = [&](int st, int it) {
        c64* a = As + st * KS * PT;
#pragma unroll
        for (int i = 0; i < (KS * PT / 2) / 256; ++i) {
            const int e = i * 256 + tid, row = e / (PT / 2), col = (e % (PT / 2)) * 2;
            const int s = it * KS + row;
            const bool ok = (s < g.N_d) && (p0 + col < g.ldp);
            cp_async16(a + row * PT + col, ok ? Abase + (long long)s * g.ldp + col : Abase, ok);
        }
    };

    c64 acc[8][4];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = mk<float>(0.f, 0.f);

    load_stage(0, 0);
    cp_async_commit();
    for (int it = 0; it < n_it; ++it) {
        cp_async_wait_all();
        __syncthreads();
        if (it + 1 < n_it) load_stage((it + 1) & 1, it + 1);
        cp_async_commit();
        const float4* a = reinterpret_cast<const float4*>(As + (it & 1) * KS * PT + ty * 8);
        const float4* d = reinterpret_cast<const float4*>(Ds + (it * KS) * NCW) + tx;
#pragma unroll
        for (int sl = 0; sl < KS; ++sl) {                  // rows beyond N_d are zero-filled tiles: they add nothing
            if (it * KS + sl >= g.N_d) break;
            const float4 d01 = d[sl * (NCW / 2)], d23 = d[sl * (NCW / 2) + NCG];
            const c64 dv[4] = {mk<float>(d01.x, d01.y), mk<float>(d01.z, d01.w), mk<float>(d23.x, d23.y),
                               mk<float>(d23.z, d23.w)};
#pragma unroll
            for (int h = 0; h < 4; ++h) {
                const float4 a2 = a[sl * (PT / 2) + h];
                const c64 a0 = mk<float>(a2.x, a2.y), a1 = mk<float>(a2.z, a2.w);
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    cmac_conj(acc[2 * h][j], a0, dv[j]);
                    cmac_conj(acc[2 * h + 1][j], a1, dv[j]);
                }
            }
        }
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const long long p = p0 + ty * 8 + i;
        if (p >= g.N_m) continue;
        c64* dst = Xout + (long long)w * g.ldx + p * g.k + r0;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int col = thread_col<NCG>(tx, j);
            if (col < kk) dst[col] = acc[i][j];
        }
    }
}

template <int TS, int TY, int NCG = 8>
cudaError_t fwd32_launch(const c64* F, const c64* X, c64* P, const GemmGeom& g, int r0, int kk, cudaStream_t s) {
    auto k = gemm32_fwd_kernel<TS, TY, NCG>;
    const size_t smem = sizeof(c64) * (2 * TY * TS * AP + 2 * KP * 4 * NCG);
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    dim3 grid((unsigned)g.split, (unsigned)g.n_f, (unsigned)((g.N_d + TY * TS - 1) / (TY * TS)));
    k<<<grid, NCG * TY, smem, s>>>(F, X, P, g, r0, kk);
    return cudaGetLastError();
}

}  // namespace

void gemm32_debug_set(int v) { g_fwd_variant = v; }

cudaError_t gemm32_fwd_launch(const void* Fhat, const void* Xhat, void* partial, const GemmGeom& g, cudaStream_t s) {
    const c64* F = static_cast<const c64*>(Fhat);
    const c64* X = static_cast<const c64*>(Xhat);
    c64* P = static_cast<c64*>(partial);
    for (int r0 = 0; r0 < g.k; r0 += NC) {
        const int kk = g.k - r0 < NC ? g.k - r0 : NC;
        cudaError_t e;
        if (kk <= 16 && g_fwd_variant == 0)   // half-width tile: 4 column groups, twice the sensor rows per CTA
            e = g.N_d <= 32 ? fwd32_launch<2, 16, 4>(F, X, P, g, r0, kk, s)
              : g.N_d <= 64 ? fwd32_launch<4, 16, 4>(F, X, P, g, r0, kk, s)
                            : fwd32_launch<8, 16, 4>(F, X, P, g, r0, kk, s);
        else if (g_fwd_variant == 1) e = g.N_d <= 32 ? fwd32_launch<1, 32>(F, X, P, g, r0, kk, s)
                                  : g.N_d <= 64 ? fwd32_launch<2, 32>(F, X, P, g, r0, kk, s)
                                                : fwd32_launch<4, 32>(F, X, P, g, r0, kk, s);
        else if (g_fwd_variant == 2) e = g.N_d <= 32 ? fwd32_launch<4, 8>(F, X, P, g, r0, kk, s)
                                       : g.N_d <= 64 ? fwd32_launch<8, 8>(F, X, P, g, r0, kk, s)
                                                     : fwd32_launch<8, 16>(F, X, P, g, r0, kk, s);
        else e = g.N_d <= 32 ? fwd32_launch<4, 8>(F, X, P, g, r0, kk, s)      // measured on B200, k = 32 (ms per launch):
               : g.N_d <= 64 ? fwd32_launch<4, 16>(F, X, P, g, r0, kk, s)     // N_d 16: 25.6 (vs 64.3 with 1 x 32 tiles),
                             : fwd32_launch<8, 16>(F, X, P, g, r0, kk, s);    // N_d 49: 45.7 (68.7), N_d 100: 72.8 (78.9)
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

cudaError_t gemm32_adj_launch(const void* Fhat, const void* Dhat, void* Xhat_out, const GemmGeom& g, cudaStream_t s) {
    for (int r0 = 0; r0 < g.k; r0 += NC) {
        const int kk = g.k - r0 < NC ? g.k - r0 : NC;
        const int ncg = kk <= 16 ? 4 : 8;
        const int PT = 8 * (256 / ncg);
        const size_t smem = sizeof(c64) * (2 * KS * PT + (size_t)g.N_d * 4 * ncg);
        if (smem > (size_t)kMaxSmem) return cudaErrorInvalidValue;   // N_d > kGemm32MaxNd: callers use the per-column path
        auto k = ncg == 4 ? gemm32_adj_kernel<4> : gemm32_adj_kernel<8>;
        cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        dim3 grid((unsigned)((g.ldp + PT - 1) / PT), (unsigned)g.n_f);
        k<<<grid, 256, smem, s>>>(static_cast<const c64*>(Fhat), static_cast<const c64*>(Dhat),
                                  static_cast<c64*>(Xhat_out), g, r0, kk);
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

}  // namespace tt
