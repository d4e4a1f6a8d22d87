/* tt_dev.h - developer hooks of libtt: test, comparison and tuning entry points that reach into the library's internals.
 * They are exported by libtt.so but are NOT part of the product ABI (include/tt.h): nothing on the path of a user's matvec
 * needs them, their signatures may change, and tt_debug_set is process-wide state meant for experiments only.
 * tests/ and bench.py use them through paper_2501_14911_b200/binding.py.  The hardware probes of bench.py live in a library
 * of their own (include/tt_probe.h, libttprobe.so). */
#ifndef TT_DEV_H_
#define TT_DEV_H_

#include "tt.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Comparison hook (bench.py's cuFFT/cuBLAS baseline reads the plan's spectrum in place instead of
 * holding a second 80 GB copy): *ptr = DEVICE address of Fhat[(w*N_d + s)*row_pitch + p], interleaved
 * complex of the plan's dtype; *row_pitch in complex elements (N_m rounded up to 16).  Read-only; valid
 * until tt_plan_destroy. */
int tt_debug_spectrum_view(const tt_plan* plan, void** ptr, int64_t* row_pitch);

/* Test hook for the planner's host logic (needs no GPU): the FFT plan of an N_t-point series.
 *   max_radix largest register butterfly allowed: 25 = the fp32 kernels' plan, 8 = the fp64 kernels' plan
 *   n_stages  receives the number of decimation-in-frequency stages
 *   radix     int[16], receives their radices (product = N_t)
 *   pos       unsigned short[N_t], pos[k] = slot of the in-place DIF output holding bin k
 *   tw        double[4*N_t], interleaved (re, im) of exp(-2 pi i k / (2 N_t)), k < 2 N_t
 * Returns TT_ERR_UNSUPPORTED_NT if N_t does not factor into {2,3,5,7} or exceeds 65535.
 * The radices are taken from {25,20,16,8,7,5,4,3,2} (those <= max_radix), largest first. */
int tt_debug_fft_tables(int64_t N_t, int max_radix, int* n_stages, int* radix, unsigned short* pos, double* tw);

/* Test hook (no GPU): the compile-time trigonometry the register butterflies use for their
 * internal twiddles, evaluated on the host: *c = cos(2 pi k / n), *s = sin(2 pi k / n). */
int tt_debug_trig(int64_t k, int64_t n, double* c, double* s);

/* Tuning hook for experiments (process-wide, affects plans created / calls made afterwards):
 * "fft_T" = series per CTA of the FFT kernels (8, 16, 32; 0 = planner's choice),
 * "fft_threads" = threads per CTA of the FFT kernels (256, 320 (inverse kernel, T = 16), 512; 0 = default), "fft_max_radix" = largest
 * register butterfly the planner may use (0 = no limit),
 * "gemv_chunk" = parameters per CTA of the forward matvec (multiple of 64; 0 = planner's choice),
 * "gemv_fwd_warps" = warps per CTA of the forward matvec (1..32; 0 = planner's choice),
 * "gemv_adj_threads" = threads per CTA of the adjoint matvec (multiple of 32, <= 512; 0 = default),
 * "fft_no_static" = 1: never use the statically specialised FFT variants (N_t = 256, 400, 500),
 * "trsv_U" = blocks of the factor in flight per warp of the triangular-solve chains (1, 2, 3; 0 = defaults),
 * "gemm32_fwd" = tile variant of the fp32 k-RHS forward GEMM (1, 2; 0 = planner's choice),
 * "gemm_adj_mt" = m-tiles per warp of the fp64 k-RHS adjoint GEMM (1, 2; 0 = default),
 * "kd_slab" = parameters per slab of the fp32 direct K assembly (multiple of 32; 0 = 8192),
 * "host_chunks" = parameter ranges of the pipelined *_host calls (1..32; 0 = planner's choice: 8 graded or 16 equal ones),
 * "l2r_mb" = F^T d with B3 as a concurrent consumer of B2: megabytes of spectrum per group of B2's grid (0 = the plain two-launch
 * sequence, -1 = planner's choice), "l2r_ctas" = its persistent consumer CTAs (0 = planner's choice), "l2r_discard" = 0 keeps the
 * write-back of the spectrum,
 * "host_growth" = size of each of those ranges in percent of the one before (1..400; 0 = planner's choice).
 * Returns TT_ERR_SHAPE for an unknown key. */
int tt_debug_set(const char* key, int value);

#ifdef __cplusplus
}
#endif
#endif /* TT_DEV_H_ */
