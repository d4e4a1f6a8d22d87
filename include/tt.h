/* tt.h - C ABI of libtt: the block lower-triangular Toeplitz parameter-to-observable
 * map F of a linear autonomous dynamical system, its transpose F^T and the normal
 * operator F^T F, applied by FFT on one NVIDIA B200 (sm_100a).
 *
 * What is computed (PAPER.md = /root/reference/PAPER.md, arxiv 2501.14911):
 *
 *   The discrete p2o map is block lower-triangular Toeplitz (eq 2.4-2.6),
 *   zero-based in time:
 *
 *        d_i = sum_{j=0..i} F_{i-j} m_j ,   i = 0..N_t-1 ,   F_k := B A^k C  (N_d x N_m)   (eq 2.5)
 *
 *   and is fully defined by its first block column F_0..F_{N_t-1}.  It is applied by
 *   embedding it in a block circulant of length L = 2 N_t that the DFT block-diagonalises
 *   (PAPER.md:263-269): zero-pad the time axis, FFT along time, one N_d x N_m complex
 *   matvec per frequency against the spectrum Fhat (computed ONCE per matrix), inverse
 *   FFT, keep the first N_t steps.  The adjoint applies the conjugate-transposed Fourier
 *   blocks of the same Fhat and is the plain Euclidean transpose
 *   (reading R2):
 *
 *        m'_j = sum_{i=j..N_t-1} F_{i-j}^T d_i ,   j = 0..N_t-1 .
 *
 *   tt_normal applies F^T F, the data-misfit Hessian of eq (2.12) with identity noise
 *   covariance.  The k-RHS calls do the same for k vectors at once
 *   (the many-matvec workloads of PAPER.md:296, 407, 421-423).
 *
 * Conventions
 *   - Every call returns TT_OK (0) or a negative tt_status; nothing throws, aborts or
 *     prints.  tt_status_string() names a code; tt_plan_last_cuda_error() returns the
 *     cudaError_t behind the last TT_ERR_CUDA / TT_ERR_OOM of a plan.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *     Apply calls only ENQUEUE work on it: no host synchronisation, no allocation
 *     (except the *_host convenience calls, see below).  A kernel fault therefore
 *     surfaces at the caller's next synchronisation.
 *   - A plan owns Fhat and its scratch buffers; the caller owns every vector and the
 *     block column (read-only, not retained).  A plan is immutable after creation but
 *     its scratch is shared: calls on one plan must be serialised (one stream, or
 *     externally ordered).
 *   - dtype TT_F32: real vectors are float, Fhat is complex64 (computed in fp64 and
 *     rounded once).  dtype TT_F64: double / complex128.
 *   - Layout TT_TIME_MAJOR is the paper's stacking:
 *        m[j*N_m + p], d[i*N_d + s], block column F[(k*N_d + s)*N_m + p];
 *     k-RHS vectors put the right-hand-side index fastest: M[(j*N_m + p)*k + r],
 *     D[(i*N_d + s)*k + r].  TT_SPACE_MAJOR (time contiguous: m[p*N_t + j], d[s*N_t + i];
 *     k-RHS M[(r*N_m + p)*N_t + j]) only changes the vectors, never the block column.
 *   - N_t must factor into {2,3,5,7} and fit the shared-memory FFT (see
 *     TT_ERR_UNSUPPORTED_NT); there is no CPU fallback of any kind.
 */
#ifndef TT_H_
#define TT_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tt_plan tt_plan;

typedef enum tt_dtype { TT_F32 = 0, TT_F64 = 1 } tt_dtype;
typedef enum tt_layout { TT_TIME_MAJOR = 0, TT_SPACE_MAJOR = 1 } tt_layout;

typedef enum tt_status {
    TT_OK = 0,
    TT_ERR_NULL = -1,           /* a required pointer is NULL */
    TT_ERR_SHAPE = -2,          /* a dimension < 1, a size overflows 63 bits, or N_d complex numbers of the plan's dtype
                                   exceed 227 KB of shared memory (N_d > 29056 for TT_F32, > 14528 for TT_F64) */
    TT_ERR_DTYPE = -3,
    TT_ERR_LAYOUT = -4,
    TT_ERR_UNSUPPORTED_NT = -5, /* N_t has a prime factor outside {2,3,5,7}, or 8 series of N_t + 1 complex128 values
                                   do not fit 227 KB of shared memory: N_t > 1815, for BOTH dtypes (the one-time
                                   transform of the matrix runs in fp64 whatever the plan's dtype) */
    TT_ERR_K = -6,              /* k < 1 or k > k_max */
    TT_ERR_ALIAS = -7,          /* out aliases in (tt_normal) */
    TT_ERR_OOM = -8,            /* cudaMalloc failed */
    TT_ERR_CUDA = -9,           /* any other CUDA runtime error (see tt_plan_last_cuda_error) */
    TT_ERR_NO_DEVICE = -10,     /* no CUDA device / wrong architecture: there is no CPU path */
    TT_ERR_NOT_SPD = -11,       /* tt_chol_create: a diagonal entry of the factor is not positive and finite */
    TT_ERR_MISMATCH = -12,      /* plans / factor / vectors of one call disagree in shape, dtype or layout */
    TT_ERR_STATIC_LIMIT = -13   /* tt_assemble_K_direct_static: the problem does not fit the library's static scratch */
} tt_status;

/* Library version, major*10000 + minor*100 + patch. */
int tt_version(void);

/* Static, NUL-terminated name of a status code. */
const char* tt_status_string(int status);

/* P0 - plan creation and the one-time DFT of the matrix ("The DFT only
 * needs to be done once for each matrix").
 *
 * For every (s,p) the series F_k[s,p], k < N_t, is zero-padded to L = 2 N_t and
 * transformed, Fhat_w[s,p] = sum_k F_k[s,p] exp(-2 pi i w k / L), keeping w = 0..N_t
 * (real input: the other half is the conjugate).  Unnormalised forward transform; the
 * 1/L sits in the inverse.
 *
 *   out                 receives the plan (set to NULL on failure)
 *   N_d, N_m, N_t       sensors, spatial parameters, time steps (all >= 1)
 *   dtype, layout       see above
 *   k_max               largest k the k-RHS calls will be given (>= 1); sizes the scratch
 *   first_block_column  [N_t][N_d][N_m] reals of `dtype`, p fastest; HOST or DEVICE pointer
 *                       (detected); read during the call, not retained
 *   stream              work is enqueued here and the call returns after it has completed
 */
int tt_plan_create(tt_plan** out, int64_t N_d, int64_t N_m, int64_t N_t, int dtype, int layout,
                   int k_max, const void* first_block_column, void* stream);

/* The same operator with its OUTPUT on a coarser time grid - the p2q map of the paper's example, whose QoIs are
 * sampled at 1 Hz while parameters and data live at 10 Hz (N_t^q = 50 << N_t = 500).
 * The paper gives no formula ("the block structure ... changes correspondingly"); reading R19: the
 * data side keeps the fine-grid steps out_every-1, 2*out_every-1, ... (the end of every out_every-th step),
 *
 *        q_I = (F m)_{out_every*(I+1)-1} ,   I = 0 .. N_t/out_every - 1 ,
 *
 * and the block column stays the fine-grid one (N_t blocks).  out_every must divide N_t.  Every data-side vector of
 * the plan (d of tt_matvec / tt_rmatvec, D of the k-RHS calls, the intermediate of tt_normal) then has
 * N_t/out_every time steps; tt_rmatvec applies the exact transpose (zeros at the steps that are not sampled).
 * The sampling and the zero-stuffing live in the load / store of the data-side FFT kernels. */
int tt_plan_create_coarse(tt_plan** out, int64_t N_d, int64_t N_m, int64_t N_t, int64_t out_every, int dtype,
                          int layout, int k_max, const void* first_block_column, void* stream);

/* Frees Fhat and all scratch.  NULL-safe.  The caller must have synchronised any stream
 * that still runs work of this plan. */
void tt_plan_destroy(tt_plan* plan);

/* Bytes of device memory the plan holds (Fhat + tables + scratch). */
size_t tt_plan_device_bytes(const tt_plan* plan);

/* cudaError_t (as int) recorded by the last failing CUDA call made for this plan; 0 if none. */
int tt_plan_last_cuda_error(const tt_plan* plan);

/* One line naming the kernels (template arguments, grid, block, shared memory) that the single-vector apply calls of this
 * plan launch for A2, B2 and the FFTs; NUL-terminated into buf[n] (TT_ERR_SHAPE if it does not fit; 512 bytes always do).
 * bench.py prints it and only quotes an ncu traffic figure whose capture names the same line. */
int tt_plan_describe(const tt_plan* plan, char* buf, size_t n);

/* Test hook: copies Fhat, unpadded, to dst_device as [N_t+1][N_d][N_m] interleaved complex
 * (complex64 for TT_F32, complex128 for TT_F64), on `stream`. */
int tt_plan_get_spectrum(const tt_plan* plan, void* dst_device, void* stream);

/* d = F m  (eq 2.5; FFT algorithm of).
 *   m  DEVICE, N_t*N_m reals, read-only;   d  DEVICE, N_t*N_d reals, overwritten. */
int tt_matvec(const tt_plan* plan, const void* m, void* d, void* stream);

/* m = F^T d  (transpose of eq 2.5; "conjugate-transposed diagonal blocks").
 *   d  DEVICE, N_t*N_d reals, read-only;   m  DEVICE, N_t*N_m reals, overwritten.
 * From ~14 GB of spectrum (and N_d >= 32) the inverse FFT of the result runs WHILE the per-frequency matvec runs, on a
 * stream owned by the plan (forked from and joined back into `stream` with events: capturable, nothing for the caller to
 * synchronise), and takes the spectrum over in the L2; the result is the two-launch sequence's bit for bit
 * (tt_plan_describe says which form a plan takes). */
int tt_rmatvec(const tt_plan* plan, const void* d, void* m, void* stream);

/* out = F^T (F m)  (eq 2.12 with Gamma_noise = I).  The intermediate
 * data vector lives in plan scratch on the device.  Between F and F^T it IS inverse
 * transformed, truncated to N_t steps, re-padded and transformed again: the truncation
 * is a projection in time that is not diagonal in frequency (reading R6).
 *   m, out  DEVICE, N_t*N_m reals; out == m returns TT_ERR_ALIAS. */
int tt_normal(const tt_plan* plan, const void* m, void* out, void* stream);

/* k-RHS variants, 1 <= k <= k_max: column r of the result equals the single-vector result
 * on column r.  The per-frequency products are complex GEMMs (N_d x N_m)(N_m x k) and
 * (N_m x N_d)(N_d x k): TT_F64 on the FP64 tensor instruction (DMMA); TT_F32 with k a multiple of 16 on the 5th-generation
 * tensor cores (tcgen05.mma kind::tf32, every fp32 product from the hi/lo tf32 parts of its factors; the adjoint for N_d <= 128),
 * any other k as register-tiled FP32 FMA GEMMs - several times slower, so callers that can choose k should take 16 or 32.
 * All three forms meet the same 1e-5 (fp32) / 1e-12 (fp64) bar against the single-vector result.
 *   M  DEVICE, N_t*N_m*k reals;   D  DEVICE, N_t*N_d*k reals (layouts above). */
int tt_matvec_batched(const tt_plan* plan, int k, const void* M, void* D, void* stream);
int tt_rmatvec_batched(const tt_plan* plan, int k, const void* D, void* M, void* stream);
/* Out = F^T (F M) for k columns at once; the intermediate data vectors live in plan scratch.  Out == M: TT_ERR_ALIAS. */
int tt_normal_batched(const tt_plan* plan, int k, const void* M, void* Out, void* stream);

/* The same calls with HOST vectors (pinned memory recommended; what bench.py's `e2e` times).  The parameter-sized
 * vector crosses PCIe in ranges of the parameter axis on a copy stream owned by the plan, overlapped with the kernels
 * of the neighbouring range on `stream` (H2D of range c+1 under the FFT + matvec of range c; D2H of range c under the
 * matvec + inverse FFT of range c+1); `stream` waits for the last copy, so synchronising it is enough.  The planner picks
 * the ranges from the shape: where the kernels of a range take longer than its copy (N_d above ~65) 8 ranges in a geometric
 * sequence with the small one at the exposed end (first for F m, last for F^T d), otherwise 16 equal ones.  Results are
 * bit-identical to the device-pointer calls.  The staging buffers, the copy stream and its events are created on first
 * use (the only apply-time allocation in the library) and freed with the plan. */
int tt_matvec_host(const tt_plan* plan, const void* m_host, void* d_host, void* stream);
int tt_rmatvec_host(const tt_plan* plan, const void* d_host, void* m_host, void* stream);
int tt_normal_host(const tt_plan* plan, const void* m_host, void* out_host, void* stream);

/* Measurement hooks (bench.py's roofline object).
 *
 * tt_plan_set_profiling(plan, 1) makes every apply call record CUDA events, on the stream
 * it launches on, around each of its kernels, and forgets earlier records; the last 64
 * profiled calls are kept.  After the caller has synchronised that stream,
 * tt_plan_stage_ms(plan, op, ms, n) returns the device time per call, averaged over the
 * recorded calls of kind `op` (a tt_op): ms[0] forward FFT of the input, ms[1] the kernel that
 * streams Fhat (per-frequency matvec / matmul), ms[2] inverse FFT (+ partial reduce),
 * ms[3] = number of calls averaged (0: nothing recorded).  TT_OP_NORMAL reports the sum of
 * its two halves.  n = number of floats ms can hold (>= 4).
 */
typedef enum tt_op {
    TT_OP_MATVEC = 0, TT_OP_RMATVEC = 1, TT_OP_NORMAL = 2, TT_OP_MATVEC_BATCHED = 3, TT_OP_RMATVEC_BATCHED = 4
} tt_op;
int tt_plan_set_profiling(tt_plan* plan, int enabled);
int tt_plan_stage_ms(const tt_plan* plan, int op, float* ms, int n);

/* ======================================================================================
 * Online phase and what Phases 2-3 of the paper need around it: the data-space
 * solve, the real-time MAP point, the SMW operator and the QoI actions.
 *
 *   G* := Gamma_prior F*  is block Toeplitz with the structure of F* when the prior is time
 *   invariant: it is the TRANSPOSE-structured operator of the block column
 *   G_k := F_k Gamma_s (N_d x N_m), i.e. a second tt_plan `G` whose tt_rmatvec applies G*.
 *   K := Gamma_noise + F G*  (eq 4.7), Gamma_noise diagonal, of order
 *   n = N_d N_t with the data stacking  row = i*N_d + s whatever the plans' layout;
 *   K = L L^T is Cholesky-factorised offline and "triangular solves are done in the online phase"
 *   (PAPER.md:294, 407).  The online inference is eq (4.13) with m_prior = 0:
 *
 *        m_map = (I - G* K^{-1} F) G* Gamma_noise^{-1} d_obs .
 * ====================================================================================== */

typedef struct tt_chol tt_chol;

/* Takes the lower Cholesky factor L of K (K = L L^T) and prepares the two triangular solves.
 *   n       order of K (>= 1)
 *   L       n x n doubles, row-major with row pitch ld (>= n) elements, HOST or DEVICE (detected);
 *           only the lower triangle is read; not retained
 *   stream  work is enqueued here and the call returns after it has completed
 * The factor is stored rescaled by the inverses of its 64 x 64 diagonal blocks (only the strictly
 * lower blocks, each contiguous, block row after block row: n^2/2 doubles) so that neither solve
 * has a diagonal solve on its dependency chain (see tt_trsv.cu).  TT_ERR_NOT_SPD if a diagonal entry is <= 0 or not finite. */
int tt_chol_create(tt_chol** out, int64_t n, const void* L, int64_t ld, void* stream);
void tt_chol_destroy(tt_chol* c);
size_t tt_chol_device_bytes(const tt_chol* c);
int tt_chol_last_cuda_error(const tt_chol* c);

/* x = K^{-1} b = L^{-T} (L^{-1} b).  b, x: DEVICE, n doubles; x may alias b.  Asynchronous on
 * `stream`, no allocation, no host synchronisation.  Calls on one tt_chol must be serialised. */
int tt_chol_solve(const tt_chol* c, const void* b, void* x, void* stream);

/* One triangular solve: transposed == 0: x = L^{-1} b;  transposed != 0: x = L^{-T} b. */
int tt_chol_trsv(const tt_chol* c, int transposed, const void* b, void* x, void* stream);

/* K = Gamma_noise + F G*, "column-by-column": columns [col0, col0 + ncols) are
 * F (G* e_c) + Gamma_noise e_c, pushed through tt_rmatvec_batched(G) and tt_matvec_batched(F) in
 * groups of min(k_max(F), k_max(G)) unit vectors.
 *   F, G       plans of identical shape, dtype and layout
 *   noise_var  DEVICE, N_t*N_d reals of the plans' dtype and layout: the diagonal of Gamma_noise
 *   K          DEVICE, n x n doubles, row-major, pitch ldk (>= n): entries K[row][c] of the requested
 *              columns are overwritten for every row; row = i*N_d + s
 * Offline call: allocates (and frees) its own scratch of N_t*(N_m + N_d)*k reals and synchronises. */
int tt_assemble_K(const tt_plan* F, const tt_plan* G, const void* noise_var, int64_t col0, int64_t ncols,
                  void* K, int64_t ldk, void* stream);

/* The same K = Gamma_noise + F G*, all of it, straight from the two block columns and without any matvec.  F is block
 * lower-triangular Toeplitz and G* = Gamma_prior F* block upper-triangular Toeplitz, so entry ((i,r),(t,s)) of
 * F G* is  sum_{j=0..min(i,t)} F_{i-j}[r,:] . G_{t-j}[s,:] : with W = Fcol Gcol^T (one real n x n x N_m GEMM of the block columns
 * seen as n x N_m matrices) it is W[(i,r),(t,s)] plus the entry one block up the block diagonal.  The paper's column-by-column
 * recipe (what tt_assemble_K does) costs 2 n FFT matvecs; this costs n^2 N_m multiply-adds (K is symmetric: the
 * lower triangle is computed, the upper one mirrored).
 *   Fcol, Gcol  DEVICE, [N_t][N_d][N_m] reals of `dtype`, N_m fastest: the first block columns F_k and G_k = F_k Gamma_prior
 *               (the arrays tt_plan_create takes with TT_TIME_MAJOR); no alignment requirement
 *   noise_var   DEVICE, [N_t][N_d] reals of `dtype`: the diagonal of Gamma_noise; NULL: K = F G* alone (see tt_K_add_noise)
 *   K           DEVICE, n x n doubles, row-major, pitch ldk (>= n), n = N_t*N_d, row = i*N_d + s; overwritten entirely
 * TT_F32: on the 5th-generation tensor cores (tcgen05.mma kind::tf32, every product from the hi/lo tf32 parts of its factors: three
 * MMAs, error <= 2^-21 per product), 128-parameter sums in tensor memory, their sums over 8192 parameters in fp32, everything
 * above that in fp64; TT_F64: fp64 throughout (FP64 tensor instruction).
 * Asynchronous on `stream`.  TT_F32 takes its scratch (the hi/lo parts of one slab of 8192 parameters of both block columns,
 * 16 n * 8192 bytes = 3.2 GB at n = 24 500) from the stream-ordered allocator (cudaMallocAsync / cudaFreeAsync on `stream`):
 * no synchronisation, TT_ERR_OOM if the device cannot provide it. */
int tt_assemble_K_direct(const void* Fcol, const void* Gcol, const void* noise_var, int64_t N_d, int64_t N_m, int64_t N_t,
                         int dtype, void* K, int64_t ldk, void* stream);

/* tt_assemble_K_direct for callers that cannot allocate (code under CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc): same arguments, same kernels, same result, TT_F32 only (TT_ERR_DTYPE otherwise - the TT_F64 path of
 * tt_assemble_K_direct has no scratch), and NO cudaMalloc / cudaMallocAsync / cudaFree or allocating library call on any path.
 * The scratch (hi / lo tf32 parts of one slab of both block columns, 16 n bytes per parameter of the slab, plus the tile list)
 * lives in a static device array of 64 MiB inside libtt.so, which every GPU that loads the library holds until the process
 * exits.  The slab is min(8192, what fits) parameters, a multiple of 32; the call returns TT_ERR_STATIC_LIMIT, having launched
 * nothing, when fewer than min(128, N_m rounded up to 32) parameters fit:
 *     16 n * 128 + 8 * ceil(n/128) * ceil(n/256) (rounded up to 256)  <=  64 MiB,   i.e. n = N_t*N_d <= ~32 700
 * (n = 24 500, the paper's shape, runs with slabs of 160 parameters: more fp64 passes over K than the 8192 of the allocating
 * call, same accuracy bound).  Smaller slabs change the fp32/fp64 summation split, so results agree with
 * tt_assemble_K_direct to rounding (~1e-6 relative), not bit for bit, unless both use the same slab.
 * All calls on a device share the one array and it keeps the previous call's contents; nothing in it needs to start at zero
 * (each slab pass rewrites what it reads).  Calls that overlap on the GPU - different streams, or graphs replayed
 * concurrently - RACE on it: serialise them.  Asynchronous on `stream`. */
int tt_assemble_K_direct_static(const void* Fcol, const void* Gcol, const void* noise_var, int64_t N_d, int64_t N_m, int64_t N_t,
                                int dtype, void* K, int64_t ldk, void* stream);

/* The N_m-sharded assembly: F G* is a SUM over parameter slices, so every rank calls
 * tt_assemble_K_direct on its own slices Fcol[:, :, P_g], Gcol[:, :, P_g] with noise_var == NULL (F G* alone), the partial
 * matrices are all-reduced (the one exchange step), and Gamma_noise (eq 4.7) is added ONCE, by this call:
 *     K[a][a] += noise_var[a],  a = 0..n-1   (noise_var: DEVICE, n reals of `dtype`, data stacking row = i*N_d + s).
 * Asynchronous on `stream`, no allocation. */
int tt_K_add_noise(const void* noise_var, int64_t n, int dtype, void* K, int64_t ldk, void* stream);

/* Phase 3 without matvecs: the data-to-QoI map Q and the QoI posterior covariance Gamma_post(q) as dense
 * matrices, from block columns.  With B = F_q G* (n_q x n) and A = F_q G_q* (n_q x n_q) - products of a block lower- with a
 * block upper-triangular Toeplitz matrix, formed like K in tt_assemble_K_direct (one GEMM of the block columns each, running sums
 * down the block diagonals; the rows (I, q) of the coarse QoI time grid are the fine-grid rows (r (I + 1) - 1, q)) -
 *     Q = F_q (I - G* K^{-1} F) G* Gamma_noise^{-1} = B K^{-1}          eq (4.11), by K - F G* = Gamma_noise
 *     Gamma_post(q) = F_q (I - G* K^{-1} F) G_q* = A - Q B^T             eq (4.10), by F G_q* = (F_q G*)^T
 * The paper obtains both by n_q operator actions each (38.4 s and ~45 s on 24 A100 for n_q = 800).
 *   Fqcol, Gqcol  DEVICE, [N_t][N_q][N_m] reals of `dtype`: block columns of the p2q map F_q on the FINE time grid and G_q,k = F_q,k Gamma_prior
 *   Gcol          DEVICE, [N_t][N_d][N_m]: G_k = F_k Gamma_prior of the p2o map
 *   out_every     r: QoIs on every r-th time step (N_t % r == 0); n_q = (N_t / r) N_q, row = I*N_q + q
 *   K             the factor of K = Gamma_noise + F G* (tt_chol_create), order n = N_t*N_d, else TT_ERR_MISMATCH
 *   Q             DEVICE, n_q x n doubles, pitch ldq (>= n);  post_cov_q: DEVICE, n_q x n_q doubles, pitch ldc (>= n_q)
 * Offline call: allocates (and frees) 8 (N_t N_q)(n + N_t N_q) + 16 n_q n + 8 n_q^2 bytes of scratch and synchronises. */
int tt_qoi_direct(const void* Fqcol, const void* Gqcol, const void* Gcol, int64_t N_q, int64_t N_d, int64_t N_m, int64_t N_t,
                  int64_t out_every, int dtype, const tt_chol* K, void* Q, int64_t ldq, void* post_cov_q, int64_t ldc,
                  void* stream);

typedef struct tt_map tt_map;
typedef enum tt_map_form {
    TT_MAP_PAPER = 0,  /* eq (4.13) as written: G*, F, K-solve, G* (footnote 14); by linearity the
                          final subtraction is done in data space:  m_map = G* (y - K^{-1} F G* y),  y = Gamma_noise^{-1} d_obs */
    TT_MAP_GAIN = 1    /* the algebraically equal gain form  m_map = G* K^{-1} d_obs  (K - F G* = Gamma_noise):
                          one G* action and one K-solve; F is not needed */
} tt_map_form;

/* Binds the operators of the online phase.  F may be NULL (then only TT_MAP_GAIN is available).
 * noise_var as in tt_assemble_K (read during the call, its reciprocal is kept).  The plans and the
 * factor are borrowed: they must outlive the tt_map.  Allocates a few data-space vectors. */
int tt_map_create(tt_map** out, const tt_plan* F, const tt_plan* G, const tt_chol* K, const void* noise_var,
                  void* stream);
void tt_map_destroy(tt_map* m);

/* m_map from the observations.  d_obs: DEVICE, N_t*N_d reals; m_map: DEVICE, N_t*N_m reals (plans' dtype
 * and layout).  Asynchronous on `stream`.  The K-solve runs in fp64 whatever the plans' dtype. */
int tt_map_infer(const tt_map* m, int form, const void* d_obs, void* m_map, void* stream);

/* out = (I - G* K^{-1} F) u : the Sherman-Morrison-Woodbury operator of eq (4.7) and eq (4.8), applied in
 * the paper's order F, K-solve, G*, subtract.  With u = Gamma_prior(m) v (the prior action is the caller's: a sparse elliptic solve
 * in the paper) it is the posterior covariance action Gamma_post(m) v, "exact up to rounding error"
 * (PAPER.md:308); with u = m_prior it is the prior-mean term m_map^prior that eq (4.13) adds.
 *   u, out  DEVICE, N_t*N_m reals (plans' dtype and layout); out == u returns TT_ERR_ALIAS.  Needs F (TT_ERR_NULL without). */
int tt_smw_apply(const tt_map* m, const void* u, void* out, void* stream);

/* Phase 3 with the p2q map: Fq and Gq are plans made by tt_plan_create_coarse from the block columns of
 * F_q and of G_q* = Gamma_prior F_q* (N_q "sensors", the same N_m, N_t, dtype and layout as the plans of `m`; any out_every).
 *   tt_postcov_q_apply:  out = Gamma_post(q) v = F_q (I - G* K^{-1} F) G_q* v            (eq 4.10)
 *                        v, out: DEVICE, (N_t/out_every)*N_q reals;  work: DEVICE, 2*N_t*N_m reals
 *   tt_d2q_apply:        q = Q d_obs = F_q m_map(d_obs), the QoI prediction of eq (4.11) / (4.14) without a stored Q;
 *                        form as in tt_map_infer;  d_obs: N_t*N_d reals;  work: N_t*N_m reals (receives m_map);  q: as v
 * Columns of Gamma_post(q) (800 x 800 in the paper) and rows of Q come from unit vectors, as in the paper. */
int tt_postcov_q_apply(const tt_map* m, const tt_plan* Fq, const tt_plan* Gq, const void* v, void* work, void* out,
                       void* stream);
int tt_d2q_apply(const tt_map* m, const tt_plan* Fq, int form, const void* d_obs, void* work, void* q, void* stream);

/* eq (4.13) in two halves, split at the one exchange step of the N_m-sharded path (DESIGN.md section 6 / 11):
 *   tt_map_infer_partial:  y = Gamma_noise^{-1} d_obs (kept in the tt_map), a = G* y -> a_scratch (N_t*N_m reals),
 *                          b = F a -> b (N_t*N_d reals).  On a rank that holds a parameter slice, b is its PARTIAL
 *                          data vector: all-reduce (sum) it over the ranks before the second half.
 *   tt_map_infer_finish:   c = K^{-1} b, m_map = G* (y - c), with the y of the preceding tt_map_infer_partial.
 *                          m_map may be the a_scratch of the first half.
 * tt_map_infer(TT_MAP_PAPER) is exactly these two calls back to back.  All pointers DEVICE, plans' dtype and layout. */
int tt_map_infer_partial(const tt_map* m, const void* d_obs, void* a_scratch, void* b, void* stream);
int tt_map_infer_finish(const tt_map* m, const void* b, void* m_map, void* stream);

/* Same with HOST vectors (pinned memory recommended): d_obs is copied in on `stream`; m_map is delivered range by range of the
 * parameter axis on the copy stream of plan G while the final G* action still computes the next range (as tt_rmatvec_host);
 * `stream` waits for the last copy. */
int tt_map_infer_host(const tt_map* m, int form, const void* d_obs_host, void* m_map_host, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* TT_H_ */
