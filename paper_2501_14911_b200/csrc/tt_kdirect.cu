// tt_kdirect.cu - tt_assemble_K_direct: K = Gamma_noise + F G* straight from the two block columns, without a single matvec.
//
// F is block lower-triangular Toeplitz with blocks F_k, G* = Gamma_prior F* block upper-triangular Toeplitz with
// blocks G_k^T, G_k = F_k Gamma_prior, so that row (i, r) of F times column (t, s) of G* is
//
//     (F G*)[(i,r),(t,s)] = sum_{j = 0 .. min(i,t)}  F_{i-j}[r,:] . G_{t-j}[s,:] .
//
// With  W[(i,r),(t,s)] = F_i[r,:] . G_t[s,:]  - ONE real GEMM  W = Fcol Gcol^T  of the block columns viewed as n x N_m matrices,
// n = N_t N_d - the sum telescopes down every block diagonal:
//
//     (F G*)[(i,r),(t,s)] = W[(i,r),(t,s)] + (F G*)[(i-1,r),(t-1,s)] .
//
// The paper forms K "column by column", one G* action and one F action per unit data vector (24 500 x 22 ms
// on 24 A100); tt_assemble_K does that with batched FFT matvecs (4.1 ms per column on one B200).  The same matrix costs
// 2 n^2 N_m flop this way (half of it: K is symmetric, only the lower triangle is computed and then mirrored) and no FFT at all.
//
//   1. W (lower tiles) = Fcol Gcol^T into K (fp64).  fp32 block columns: kd_umma_kernel (tt_kdirect_umma.cu) - tcgen05.mma
//                         kind::tf32 with the 3-product hi/lo split, TMA-fed, accumulators in tensor memory.  fp64 block
//                         columns: kd_gemm_dmma_kernel, the FP64 tensor instruction (tcgen05 has no f64 kind)
//   2. kd_diag_kernel     in-place running sums down the block diagonals of the lower triangle, + Gamma_noise on the diagonal
//   3. kd_mirror_kernel   upper triangle := transpose of the lower one
//
// Precision: TT_F32 forms every product from the tf32 hi/lo parts of its factors (error <= 2^-21 per product), sums 128
// parameters in the tensor core's fp32 accumulator, the 128-parameter sums of a slab of 8192 in fp32 registers, and the slab
// sums and the running sums of step 2 in fp64; TT_F64 is fp64 throughout (DMMA).
#include <type_traits>

#include "../../include/tt.h"
#include "tt_common.cuh"
#include "tt_internal.h"

namespace tt {
namespace {

constexpr int kKdBM = 128;     // rows of Fcol per CTA tile (fp64 DMMA kernel)
constexpr int kKdBK = 32;      // parameters per shared-memory stage
constexpr int kKdThreads = 256;

// fp64 on the FP64 tensor pipe: mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4), the same instruction as the k-RHS GEMMs of tt_gemm.cu.
// CTA tile 128 x 64, 8 warps as 4 x 2, warp tile 32 x 32 = 4 x 4 DMMA tiles; stages of 32 parameters read with scalar loads (rows have no alignment); the [row][k] tile has
// a pitch of 36 doubles, so the fragment loads (row lane/4, k lane%4) of each half-warp fall into 16 different 8-byte bank pairs.
// A fragment: A[row = lane/4][k = lane%4]; B fragment: B[n = lane/4][k = lane%4]; C: [lane/4][2 (lane%4) + {0, 1}].
__device__ __forceinline__ void kd_dmma(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
constexpr int kKdDmmaBN = 64, kKdDmmaP = kKdBK + 4;
__global__ void __launch_bounds__(kKdThreads, 1)
kd_gemm_dmma_kernel(const double* __restrict__ A, const double* __restrict__ B, double* __restrict__ C, const long long nA,
                    const long long nB, const long long Kdim, const long long ldc, const int lower_only) {
    constexpr int P = kKdDmmaP, BN = kKdDmmaBN, ROWS = kKdBM + BN, LA = kKdBM / 8, LB = BN / 8;
    const int tn = blockIdx.x, tm = blockIdx.y;
    if (lower_only && (long long)tn * BN >= (long long)(tm + 1) * kKdBM) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double* sm = reinterpret_cast<double*>(smem_raw);   // [2][ROWS][P]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, tq = lane & 3;
    const int wm = warp >> 1, wn = warp & 1;
    const long long rowA0 = (long long)tm * kKdBM, rowB0 = (long long)tn * BN;
    const double* pa = A + (rowA0 + warp) * Kdim + lane;
    const double* pb = B + (rowB0 + warp) * Kdim + lane;
    unsigned okA = 0, okB = 0;
#pragma unroll
    for (int i = 0; i < LA; ++i) okA |= (rowA0 + warp + 8 * i < nA ? 1u : 0u) << i;
#pragma unroll
    for (int i = 0; i < LB; ++i) okB |= (rowB0 + warp + 8 * i < nB ? 1u : 0u) << i;
    double pre[LA + LB];
    auto gload = [&](long long k0) {
        const bool kok = k0 + lane < Kdim;
#pragma unroll
        for (int i = 0; i < LA; ++i) pre[i] = (kok && ((okA >> i) & 1u)) ? __ldg(pa + k0 + (long long)(8 * i) * Kdim) : 0.0;
#pragma unroll
        for (int i = 0; i < LB; ++i) pre[LA + i] = (kok && ((okB >> i) & 1u)) ? __ldg(pb + k0 + (long long)(8 * i) * Kdim) : 0.0;
    };
    auto sstore = [&](int stage) {
        double* s = sm + stage * (ROWS * P);
#pragma unroll
        for (int i = 0; i < LA; ++i) s[(warp + 8 * i) * P + lane] = pre[i];
#pragma unroll
        for (int i = 0; i < LB; ++i) s[(kKdBM + warp + 8 * i) * P + lane] = pre[LA + i];
    };
    double acc[4][4][2];
#pragma unroll
    for (int mt = 0; mt < 4; ++mt)
#pragma unroll
        for (int nt = 0; nt < 4; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = 0.0;
    const int nk = (int)((Kdim + kKdBK - 1) / kKdBK);
    gload(0);
    sstore(0);
    __syncthreads();
    for (int t = 0; t < nk; ++t) {
        if (t + 1 < nk) gload((long long)(t + 1) * kKdBK);
        const double* s = sm + (t & 1) * (ROWS * P);
        const double* sa = s + (wm * 32 + g) * P + tq;
        const double* sb = s + (kKdBM + wn * 32 + g) * P + tq;
#pragma unroll
        for (int k4 = 0; k4 < kKdBK / 4; ++k4) {
            double a[4], b[4];
#pragma unroll
            for (int mt = 0; mt < 4; ++mt) a[mt] = sa[mt * 8 * P + k4 * 4];
#pragma unroll
            for (int nt = 0; nt < 4; ++nt) b[nt] = sb[nt * 8 * P + k4 * 4];
#pragma unroll
            for (int mt = 0; mt < 4; ++mt)
#pragma unroll
                for (int nt = 0; nt < 4; ++nt) kd_dmma(acc[mt][nt][0], acc[mt][nt][1], a[mt], b[nt]);
        }
        if (t + 1 < nk) sstore((t + 1) & 1);
        __syncthreads();
    }
#pragma unroll
    for (int mt = 0; mt < 4; ++mt)
#pragma unroll
        for (int nt = 0; nt < 4; ++nt)
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                const long long row = rowA0 + wm * 32 + mt * 8 + g, col = rowB0 + wn * 32 + nt * 8 + 2 * tq + r;
                if (row < nA && col < nB) C[row * ldc + col] = acc[mt][nt][r];
            }
}

// Lower triangle, in place: K[a][b] := sum_{j >= 0} W[a - j N_d][b - j N_d]  (+ noise_var[a] if a == b; noise_var may be null).  One thread per
// chain = per start (a0, b0) in the first block column (b0 < N_d, a0 >= b0); consecutive threads are consecutive b0.
template <typename R>
__global__ void __launch_bounds__(256)
kd_diag_kernel(double* __restrict__ K, const R* __restrict__ noise_var, const long long n, const int N_d,
               const long long ldk) {
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long a0 = idx / N_d;
    const int b0 = (int)(idx - a0 * N_d);
    if (a0 >= n || b0 > a0) return;
    double run = 0.0;
    long long a = a0, b = b0;
    for (; a < n; a += N_d, b += N_d) {
        double* p = K + a * ldk + b;
        run += *p;
        *p = (a == b && noise_var) ? run + (double)noise_var[a] : run;
    }
}

// K[b][a] := K[a][b] for a > b, through 32 x 32 shared-memory tiles
__global__ void __launch_bounds__(256)
kd_mirror_kernel(double* __restrict__ K, const long long n, const long long ldk) {
    __shared__ double tile[32][33];
    const int tj = blockIdx.x, ti = blockIdx.y;
    if (tj > ti) return;
    const int x = threadIdx.x & 31, y0 = threadIdx.x >> 5;
    for (int y = y0; y < 32; y += 8) {
        const long long a = (long long)ti * 32 + y, b = (long long)tj * 32 + x;
        tile[y][x] = (a < n && b < n) ? K[a * ldk + b] : 0.0;
    }
    __syncthreads();
    for (int y = y0; y < 32; y += 8) {
        const long long b = (long long)tj * 32 + y, a = (long long)ti * 32 + x;   // writes K[b][a], a fastest
        if (a < n && b < n && a > b) K[b * ldk + a] = tile[x][y];
    }
}

// C (nA x nB, fp64, pitch ldc) = A B^T for row-major A (nA x Kdim) and B (nB x Kdim) of type R; lower_only: only the tiles that
// touch the lower triangle (nA == nB)
template <typename R>
cudaError_t kd_launch_gemm(const R* A, const R* B, double* C, long long nA, long long nB, long long Kdim, long long ldc,
                           int lower_only, cudaStream_t s) {
    cudaError_t e = cudaSuccess;
    if constexpr (sizeof(R) == 8) {   // DMMA: 0.585 s against 0.864 s for a register-tiled DFMA form at N_m = 26 316
        const size_t smem = (size_t)2 * (kKdBM + kKdDmmaBN) * kKdDmmaP * sizeof(double);
        e = cudaFuncSetAttribute(kd_gemm_dmma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        const dim3 grid((unsigned)((nB + kKdDmmaBN - 1) / kKdDmmaBN), (unsigned)((nA + kKdBM - 1) / kKdBM));
        kd_gemm_dmma_kernel<<<grid, kKdThreads, smem, s>>>(A, B, C, nA, nB, Kdim, ldc, lower_only);
    } else {   // fp32: 3 x tf32 split on tcgen05 (tt_kdirect_umma.cu)
        return kd_umma_gemm(A, B, C, nA, nB, Kdim, ldc, lower_only, s);
    }
    return cudaGetLastError();
}

template <typename R>
cudaError_t kd_run(const R* Fcol, const R* Gcol, const R* noise_var, long long N_d, long long N_m, long long N_t, double* K,
                   long long ldk, cudaStream_t s) {
    const long long n = N_t * N_d;
    cudaError_t e = kd_launch_gemm<R>(Fcol, Gcol, K, n, n, N_m, ldk, 1, s);
    if (e != cudaSuccess) return e;
    const long long chains = n * N_d;
    kd_diag_kernel<R><<<(unsigned)((chains + 255) / 256), 256, 0, s>>>(K, noise_var, n, (int)N_d, ldk);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    const unsigned nt = (unsigned)((n + 31) / 32);
    kd_mirror_kernel<<<dim3(nt, nt), 256, 0, s>>>(K, n, ldk);
    return cudaGetLastError();
}

// Whole matrix, in place: M[a][b] := sum_{j >= 0} W[a - j sa][b - j sb] (the block rows of the two operands may differ in
// height).  One thread per chain; a chain starts in the first block column (b0 < sb) or in the first block row (a0 < sa).
__global__ void __launch_bounds__(256)
kd_diag_rect_kernel(double* __restrict__ M, const long long nA, const long long nB, const int sa, const int sb,
                    const long long ld) {
    long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long first = nA * sb;
    long long a0, b0;
    if (idx < first) {
        a0 = idx / sb;
        b0 = idx - a0 * sb;
    } else {
        idx -= first;
        const long long wb = nB - sb;
        if (wb <= 0) return;
        a0 = idx / wb;
        if (a0 >= sa) return;
        b0 = sb + (idx - a0 * wb);
    }
    if (a0 >= nA || b0 >= nB) return;
    double run = 0.0;
    for (long long a = a0, b = b0; a < nA && b < nB; a += sa, b += sb) {
        double* p = M + a * ld + b;
        run += *p;
        *p = run;
    }
}

// dst[ro][co] = src[rmap(ro)][cmap(co)]: rows / columns (I, q) of a coarse time grid are the fine-grid rows (r (I + 1) - 1, q)
// (reading R19); r == 1: identity
__global__ void __launch_bounds__(256)
kd_pick_kernel(const double* __restrict__ src, const long long lds, double* __restrict__ dst, const long long ldd,
               const long long nro, const long long nco, const int Nr, const int rr, const int Nc, const int rc) {
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= nro * nco) return;
    const long long ro = idx / nco, co = idx - ro * nco;
    const long long rs = rr > 1 ? ((long long)rr * (ro / Nr + 1) - 1) * Nr + ro % Nr : ro;
    const long long cs = rc > 1 ? ((long long)rc * (co / Nc + 1) - 1) * Nc + co % Nc : co;
    dst[ro * ldd + co] = src[rs * lds + cs];
}

// out[i][j] -= c[i][j]
__global__ void __launch_bounds__(256)
kd_sub_kernel(double* __restrict__ out, const long long ldo, const double* __restrict__ c, const long long ldc,
              const long long nr, const long long nc) {
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= nr * nc) return;
    const long long i = idx / nc, j = idx - i * nc;
    out[i * ldo + j] -= c[i * ldc + j];
}

struct KdScratch {   // frees on every exit path
    void* p[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
    ~KdScratch() { for (void* q : p) if (q) cudaFree(q); }
};

template <typename R>
int kd_qoi_run(const R* Fq, const R* Gq, const R* G, long long N_q, long long N_d, long long N_m, long long N_t, long long r,
               const ::tt_chol* K, double* Q, long long ldq, double* pcq, long long ldc, cudaStream_t s) {
    const long long nqf = N_t * N_q, n = N_t * N_d, nq = (N_t / r) * N_q;
    KdScratch ws;
    double *Bfull, *Afull, *Bdec, *Qc, *Cq;
    cudaError_t e = cudaMalloc(&ws.p[0], (size_t)nqf * n * 8);
    if (e == cudaSuccess) e = cudaMalloc(&ws.p[1], (size_t)nqf * nqf * 8);
    if (e == cudaSuccess) e = cudaMalloc(&ws.p[2], (size_t)nq * n * 8);
    if (e == cudaSuccess) e = cudaMalloc(&ws.p[3], (size_t)nq * n * 8);
    if (e == cudaSuccess) e = cudaMalloc(&ws.p[4], (size_t)nq * nq * 8);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return TT_ERR_OOM; }
    Bfull = static_cast<double*>(ws.p[0]); Afull = static_cast<double*>(ws.p[1]); Bdec = static_cast<double*>(ws.p[2]);
    Qc = static_cast<double*>(ws.p[3]); Cq = static_cast<double*>(ws.p[4]);
#define KD_TRY(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { (void)cudaGetLastError(); return TT_ERR_CUDA; } } while (0)
    auto blocks = [](long long work) { return (unsigned)((work + 255) / 256); };
    // B = F_q G* on the fine grid, then its coarse rows
    KD_TRY(kd_launch_gemm<R>(Fq, G, Bfull, nqf, n, N_m, n, 0, s));
    kd_diag_rect_kernel<<<blocks(nqf * N_d + N_q * (n - N_d)), 256, 0, s>>>(Bfull, nqf, n, (int)N_q, (int)N_d, n);
    KD_TRY(cudaGetLastError());
    kd_pick_kernel<<<blocks(nq * n), 256, 0, s>>>(Bfull, n, Bdec, n, nq, n, (int)N_q, (int)r, (int)N_d, 1);
    KD_TRY(cudaGetLastError());
    // A = F_q G_q* on the fine grid, then its coarse rows and columns, straight into the output
    // (symmetric like K: lower tiles, running sums on the lower triangle, mirror)
    KD_TRY(kd_launch_gemm<R>(Fq, Gq, Afull, nqf, nqf, N_m, nqf, 1, s));
    kd_diag_kernel<R><<<blocks(nqf * N_q), 256, 0, s>>>(Afull, static_cast<const R*>(nullptr), nqf, (int)N_q, nqf);
    KD_TRY(cudaGetLastError());
    kd_mirror_kernel<<<dim3((unsigned)((nqf + 31) / 32), (unsigned)((nqf + 31) / 32)), 256, 0, s>>>(Afull, nqf, nqf);
    KD_TRY(cudaGetLastError());
    kd_pick_kernel<<<blocks(nq * nq), 256, 0, s>>>(Afull, nqf, pcq, ldc, nq, nq, (int)N_q, (int)r, (int)N_q, (int)r);
    KD_TRY(cudaGetLastError());
    // Q = B K^{-1}: K is symmetric, so row i of Q is K^{-1} (row i of B)
    for (long long i = 0; i < nq; ++i) {
        const int st = tt_chol_solve(K, Bdec + i * n, Qc + i * n, s);
        if (st != TT_OK) return st;
    }
    KD_TRY(cudaMemcpy2DAsync(Q, (size_t)ldq * 8, Qc, (size_t)n * 8, (size_t)n * 8, (size_t)nq, cudaMemcpyDeviceToDevice, s));
    // Gamma_post(q) = A - Q B^T
    KD_TRY(kd_launch_gemm<double>(Qc, Bdec, Cq, nq, nq, n, nq, 0, s));
    kd_sub_kernel<<<blocks(nq * nq), 256, 0, s>>>(pcq, ldc, Cq, nq, nq, nq);
    KD_TRY(cudaGetLastError());
    KD_TRY(cudaStreamSynchronize(s));   // the scratch is freed on return
#undef KD_TRY
    return TT_OK;
}

}  // namespace
}  // namespace tt

extern "C" int tt_assemble_K_direct(const void* Fcol, const void* Gcol, const void* noise_var, int64_t N_d, int64_t N_m,
                                    int64_t N_t, int dtype, void* K, int64_t ldk, void* stream) {
    using namespace tt;
    if (!Fcol || !Gcol || !K) return TT_ERR_NULL;   // noise_var == NULL: F G* alone (a rank's partial sum of the sharded assembly)
    if (dtype != TT_F32 && dtype != TT_F64) return TT_ERR_DTYPE;
    if (N_d < 1 || N_m < 1 || N_t < 1 || N_d > 65535) return TT_ERR_SHAPE;
    const long long n = N_d * N_t;
    if (ldk < n || n > (1LL << 24)) return TT_ERR_SHAPE;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { (void)cudaGetLastError(); return TT_ERR_NO_DEVICE; }
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        (void)cudaGetLastError();
        return TT_ERR_NO_DEVICE;
    }
    if (prop.major != 10) return TT_ERR_NO_DEVICE;   // built for sm_100a only
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    cudaError_t e = dtype == TT_F32
        ? kd_run<float>(static_cast<const float*>(Fcol), static_cast<const float*>(Gcol), static_cast<const float*>(noise_var),
                           N_d, N_m, N_t, static_cast<double*>(K), ldk, s)
        : kd_run<double>(static_cast<const double*>(Fcol), static_cast<const double*>(Gcol),
                            static_cast<const double*>(noise_var), N_d, N_m, N_t, static_cast<double*>(K), ldk, s);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return e == cudaErrorMemoryAllocation ? TT_ERR_OOM : TT_ERR_CUDA; }
    return TT_OK;
}

// tt_assemble_K_direct for TT_F32 without any allocation: the same kernels, the GEMM's scratch in a static device array
// (kd_umma_gemm_static, tt_kdirect_umma.cu).
extern "C" int tt_assemble_K_direct_static(const void* Fcol, const void* Gcol, const void* noise_var, int64_t N_d, int64_t N_m,
                                           int64_t N_t, int dtype, void* K, int64_t ldk, void* stream) {
    using namespace tt;
    if (!Fcol || !Gcol || !K) return TT_ERR_NULL;
    if (dtype != TT_F32) return TT_ERR_DTYPE;        // the TT_F64 path of tt_assemble_K_direct has no scratch to begin with
    if (N_d < 1 || N_m < 1 || N_t < 1 || N_d > 65535) return TT_ERR_SHAPE;
    const long long n = N_d * N_t;
    if (ldk < n || n > (1LL << 24)) return TT_ERR_SHAPE;
    int dev = 0, major = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) {
        (void)cudaGetLastError();
        return TT_ERR_NO_DEVICE;
    }
    if (major != 10) return TT_ERR_NO_DEVICE;   // built for sm_100a only
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    double* Kd = static_cast<double*>(K);
    int fits = 0;
    cudaError_t e = kd_umma_gemm_static(static_cast<const float*>(Fcol), static_cast<const float*>(Gcol), Kd, n, n, N_m, ldk, 1, s, &fits);
    if (e == cudaSuccess && !fits) return TT_ERR_STATIC_LIMIT;
    if (e == cudaSuccess) {
        const long long chains = n * N_d;
        kd_diag_kernel<float><<<(unsigned)((chains + 255) / 256), 256, 0, s>>>(Kd, static_cast<const float*>(noise_var), n, (int)N_d, ldk);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) {
        const unsigned nt = (unsigned)((n + 31) / 32);
        kd_mirror_kernel<<<dim3(nt, nt), 256, 0, s>>>(Kd, n, ldk);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) { (void)cudaGetLastError(); return TT_ERR_CUDA; }
    return TT_OK;
}

// K[a][a] += noise_var[a]
template <typename R>
__global__ void __launch_bounds__(256)
kd_add_noise_kernel(double* __restrict__ K, const R* __restrict__ noise_var, const long long n, const long long ldk) {
    const long long a = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (a < n) K[a * ldk + a] += (double)noise_var[a];
}

extern "C" int tt_K_add_noise(const void* noise_var, int64_t n, int dtype, void* K, int64_t ldk, void* stream) {
    if (!noise_var || !K) return TT_ERR_NULL;
    if (dtype != TT_F32 && dtype != TT_F64) return TT_ERR_DTYPE;
    if (n < 1 || ldk < n) return TT_ERR_SHAPE;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const unsigned nb = (unsigned)((n + 255) / 256);
    if (dtype == TT_F32) kd_add_noise_kernel<float><<<nb, 256, 0, s>>>(static_cast<double*>(K), static_cast<const float*>(noise_var), n, ldk);
    else kd_add_noise_kernel<double><<<nb, 256, 0, s>>>(static_cast<double*>(K), static_cast<const double*>(noise_var), n, ldk);
    if (cudaGetLastError() != cudaSuccess) return TT_ERR_CUDA;
    return TT_OK;
}

extern "C" int tt_qoi_direct(const void* Fqcol, const void* Gqcol, const void* Gcol, int64_t N_q, int64_t N_d, int64_t N_m,
                             int64_t N_t, int64_t out_every, int dtype, const tt_chol* K, void* Q, int64_t ldq,
                             void* post_cov_q, int64_t ldc, void* stream) {
    using namespace tt;
    if (!Fqcol || !Gqcol || !Gcol || !K || !Q || !post_cov_q) return TT_ERR_NULL;
    if (dtype != TT_F32 && dtype != TT_F64) return TT_ERR_DTYPE;
    if (N_q < 1 || N_d < 1 || N_m < 1 || N_t < 1 || out_every < 1 || N_t % out_every != 0 || N_q > 65535 || N_d > 65535)
        return TT_ERR_SHAPE;
    const long long n = N_d * N_t, nq = (N_t / out_every) * N_q;
    if (ldq < n || ldc < nq || n > (1LL << 24) || N_t * N_q > (1LL << 24)) return TT_ERR_SHAPE;
    if (chol_order(K) != n) return TT_ERR_MISMATCH;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { (void)cudaGetLastError(); return TT_ERR_NO_DEVICE; }
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        (void)cudaGetLastError();
        return TT_ERR_NO_DEVICE;
    }
    if (prop.major != 10) return TT_ERR_NO_DEVICE;   // built for sm_100a only
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (dtype == TT_F32)
        return kd_qoi_run<float>(static_cast<const float*>(Fqcol), static_cast<const float*>(Gqcol), static_cast<const float*>(Gcol),
                                 N_q, N_d, N_m, N_t, out_every, K, static_cast<double*>(Q), ldq, static_cast<double*>(post_cov_q), ldc, s);
    return kd_qoi_run<double>(static_cast<const double*>(Fqcol), static_cast<const double*>(Gqcol), static_cast<const double*>(Gcol),
                              N_q, N_d, N_m, N_t, out_every, K, static_cast<double*>(Q), ldq, static_cast<double*>(post_cov_q), ldc, s);
}
