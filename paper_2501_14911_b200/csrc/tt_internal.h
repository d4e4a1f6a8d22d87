// tt_internal.h - host-side declarations shared by the libtt translation units.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

struct tt_plan;
struct tt_chol;

namespace tt {

// What the online-phase calls (tt_online.cu) need to know about a plan.
struct PlanInfo {
    long long N_d, N_m, N_t;
    int dtype, layout, k_max;
    long long dec;  // data vectors on every dec-th time step (tt_plan_create_coarse)
};
PlanInfo plan_info(const ::tt_plan* p);
long long chol_order(const ::tt_chol* c);  // order n of the factor (tt_online.cu)
// m_host = F^T d_dev, delivered to HOST memory with the D2H copies pipelined behind the kernels (tt_api.cu); returns a tt_status
int plan_rmatvec_to_host(const ::tt_plan* p, const void* d_dev, void* m_host, cudaStream_t s);

constexpr int kMaxStages = 16;
constexpr int kMaxSmem = 232448;  // 227 KB: largest dynamic shared memory per CTA on sm_100

// Geometry of one batched 1-D FFT launch along time.  A "series" is one time series of
// N_t reals; the transforms use the packed real-FFT trick, i.e. one N-point complex FFT
// (N = N_t) of z_n = x_{2n} + i x_{2n+1} stands for the L = 2N-point real FFT of the
// zero-padded series.
//
// Element addresses (in elements of the respective type), series b in [0,B), y = blockIdx.y:
//   real side    : real[y*r_ys + b*r_bs + j*r_ts]              j = 0..N-1   (time step)
//   complex side : cplx[y*c_ys + b*c_bs + w*c_fs (+ c*c_ps)]    w = 0..N     (frequency)
struct FftParams {
    int N;                  // complex FFT length = N_t
    int n_stages;
    int radix[kMaxStages];  // product = N, applied in order as decimation-in-frequency passes;
                            // each from {2,3,4,5,7,8,16,20,25}
    unsigned magic[kMaxStages];  // ceil(2^32 / M_st), M_st = block length after pass st (exact u / M_st for u < 2^16)
    const void* tw;         // Cx<Tc>[2N]: tw[k] = exp(-2 pi i k / (2N))
    const unsigned short* pos;  // pos[k] = slot of the in-place DIF output that holds bin k, k < N; followed by the
                                // inverse table: pos[N + slot] = bin held by that slot
    long long B;            // series per y-row
    long long B_store;      // forward only: series in [B, B_store) are stored as zeros (row padding)
    long long r_ys, r_bs, r_ts;
    long long c_ys, c_bs, c_fs;
    double scale;           // inverse only: factor applied to the real output (1/L)
    int discard_in;         // consumer kernel only: drop the input lines from the L2 once read (no write-back)
    const unsigned char* skip;  // inverse only: tiles (CTAs) whose flag is set have been done by the consumer kernel: exit at once
    int dec;                // real side on a coarser time grid: only the time steps j with (j+1) % dec == 0 exist, stored
                            // at index (j+1)/dec - 1 (forward: the others are zeros; inverse: the others are dropped); 1 = all
};

struct FftChoice {
    int T;        // series per CTA
    int threads;  // threads per CTA
    size_t smem;  // dynamic shared memory bytes
};
// elem = sizeof(Cx<Tc>); returns T = 0 if even T = 8 does not fit.
FftChoice fft_choose(int N, size_t elem);

// tin/tc/tout: 0 = float, 1 = double.  ny = gridDim.y.
cudaError_t fft_r2c_launch(int tin, int tc, int tout, const void* real_in, void* cplx_out,
                           const FftParams& P, int ny, cudaStream_t s);
cudaError_t fft_c2r_launch(int tc, const void* cplx_in, void* real_out, const FftParams& P, int ny,
                           cudaStream_t s);
// B3 as persistent consumer of a running B2 (tt_fft.cu fft_c2r_consumer_kernel): sync = [ticket, error, counters per ptile parameters]
bool fft_c2r_consumer_ok(int tc, int N, int ptile);
cudaError_t fft_c2r_consumer_launch(int tc, const void* cplx_in, void* real_out, const FftParams& P, unsigned* sync,
                                    unsigned char* done, int ptile, int n_ctas, cudaStream_t s);
// dhat[w*N_d + s] = sum_c partial[(w*n_chunks + c)*N_d + s] (fixed order, fp64 accumulator)
cudaError_t reduce_partials_launch(int dt, const void* partial, void* dhat, int n_f, int n_chunks, int N_d,
                                   cudaStream_t s);
void fft_debug_force_T(int T);  // 0 = planner's choice
void fft_debug_force_threads(int NT);  // 256 or 512; 0 = default (512 for fp32, 256 for fp64)
void fft_debug_no_static(int v);  // 1 = never use the statically specialised FFT variants
double debug_cos2pi(long long k, long long n);
double debug_sin2pi(long long k, long long n);

// Per-frequency matvecs.  Fhat[(w*N_d + s)*ldp + p], xhat[w*ldp + p], dhat[w*N_d + s];
// partial[(w*n_chunks + c)*N_d + s] = sum over chunk c of Fhat_w[s,:] xhat_w[:].
struct GemvGeom {
    int n_f;        // N_t + 1 frequencies
    int N_d;
    long long ldp;  // padded N_m (multiple of 16 elements)
    int chunk;      // forward: elements of p per CTA (multiple of 64)
    int n_chunks;
    int warps;      // forward: warps per CTA (0 = kernel default)
    unsigned* l2r_sync = nullptr;  // adjoint, producer mode (with B3 as consumer): [ticket, error, one counter per CTA tile of parameters]
    int l2r_tpg = 0;               // producer mode: CTA tiles per group - the grid runs group by group, all frequencies of a group before the next
    long long p_begin = 0, p_end = 0;  // restrict the launch to parameters [p_begin, p_end) (p_end == 0: all); p_begin must be
                                       // a multiple of `chunk` (forward) and of 512 (adjoint) - the pipelined *_host calls
};
void gemv_debug_set(int fwd_warps, int adj_threads);  // -1 = leave, 0 = planner's choice
cudaError_t gemv_fwd_launch(int dt, const void* Fhat, const void* xhat, void* partial, const GemvGeom& g,
                            cudaStream_t s);
cudaError_t gemv_adj_launch(int dt, const void* Fhat, const void* dhat, void* xhat_out, const GemvGeom& g,
                            cudaStream_t s);
int gemv_adj_tile_params(int dt);  // parameters per CTA of the adjoint kernel (the granularity of the producer-mode counters)
int gemv_describe(int dt, const GemvGeom& g, char* buf, size_t n);  // snprintf semantics

// k-RHS per-frequency complex GEMMs on the FP64 tensor pipe (DMMA) / fp32 FMA.
//   Xhat[(w*N_m_pad... see tt_gemm.cu
struct GemmGeom {
    int n_f, N_d, k;
    long long N_m, ldp;     // Fhat row pitch
    long long ldx;          // Xhat pitch per frequency: Xhat[w*ldx + p*k + r]
    int split;              // forward: number of p-splits (partials)
    long long p_per_split;
};
cudaError_t gemm_fwd_launch(int dt, const void* Fhat, const void* Xhat, void* partial, const GemmGeom& g,
                            cudaStream_t s);
cudaError_t gemm_adj_launch(int dt, const void* Fhat, const void* Dhat, void* Xhat_out, const GemmGeom& g,
                            cudaStream_t s);

void gemm_debug_set_adj(int m_tiles_per_warp);  // 1 or 2 (default)

// complex64 FMA GEMMs of TT_F32 plans (tt_gemm32.cu); N_d <= kGemm32MaxNd for the adjoint (Dhat_w lives in shared memory)
constexpr int kGemm32MaxNd = 768;
cudaError_t gemm32_fwd_launch(const void* Fhat, const void* Xhat, void* partial, const GemmGeom& g, cudaStream_t s);
cudaError_t gemm32_adj_launch(const void* Fhat, const void* Dhat, void* Xhat_out, const GemmGeom& g, cudaStream_t s);
void gemm32_debug_set(int fwd_variant);
// the same products on tcgen05 (3xTF32, tt_gemm32_umma.cu) for the shapes *_ok() accepts
bool gemm32_umma_fwd_ok(const GemmGeom& g);
cudaError_t gemm32_umma_fwd_launch(const void* Fhat, const void* Xhat, void* partial, const GemmGeom& g, cudaStream_t s);
bool gemm32_umma_adj_ok(const GemmGeom& g);
cudaError_t gemm32_umma_adj_launch(const void* Fhat, const void* Dhat, void* Xhat_out, const GemmGeom& g, cudaStream_t s);
void gemm32_umma_debug_set(int enable);

// Triangular solves with the rescaled Cholesky factor (tt_trsv.cu).
constexpr int kTrsvNB = 64;  // block order
struct TrsvGeom {
    long long n;       // order of K
    int nblk;          // ceil(n / kTrsvNB)
    const double* Lt;  // strictly-lower blocks of D^{-1} L, block (I,J) contiguous at NB*NB*(I*(I-1)/2 + J)
    const double* Dinv;  // [nblk][NB][NB] inverses of the diagonal blocks (identity on the padding)
    double* bt;        // [nblk*NB] D^{-1} b
    double* y;         // [nblk*NB] forward solution (self-flagging)
    double* xt;        // [nblk*NB] backward solution before the D^{-T} post-step (self-flagging)
    unsigned* ticket;  // [2] block tickets of the forward / backward chain
};
// Plan time: D_I^{-1} and Lt for the block rows of the slab src = rows [row0, row0 + nrows) of the row-major
// factor (pitch ld), row0 a multiple of kTrsvNB; *bad is set to 1 if a diagonal entry is not positive and finite.
cudaError_t trsv_prepare_launch(const double* src, long long ld, long long row0, long long nrows, long long n,
                                double* Dinv, double* Lt, int* bad, cudaStream_t s);
cudaError_t trsv_pre_launch(const TrsvGeom& g, const double* b, cudaStream_t s);   // bt = D^{-1} b (b may be null), resets
cudaError_t trsv_fwd_launch(const TrsvGeom& g, cudaStream_t s);                    // y = Lt^{-1} bt
cudaError_t trsv_bwd_launch(const TrsvGeom& g, const double* yin, cudaStream_t s); // xt = Lt^{-T} yin
cudaError_t trsv_post_launch(const TrsvGeom& g, double* x, cudaStream_t s);        // x = D^{-T} xt
void trsv_debug_set_U(int U);  // blocks in flight per warp: 1, 2 (default), 3
cudaError_t trsv_copy_launch(const double* src, double* dst, long long n, cudaStream_t s);

// fp32 C (fp64) = A B^T on tcgen05 (3 x tf32 split, TMA-fed, accumulators in tensor memory): tt_kdirect_umma.cu
cudaError_t kd_umma_gemm(const float* A, const float* B, double* C, long long nA, long long nB, long long Kdim, long long ldc,
                         int lower_only, cudaStream_t s);
// the same with the scratch in a static device array (no allocation); *fits = 0 and no launch if the problem is too large for it
cudaError_t kd_umma_gemm_static(const float* A, const float* B, double* C, long long nA, long long nB, long long Kdim, long long ldc,
                                int lower_only, cudaStream_t s, int* fits);
void kd_umma_debug_set_slab(int ks);  // parameters accumulated in tensor memory between fp64 flushes (0 = default)


}  // namespace tt
