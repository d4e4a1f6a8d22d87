/* tt_probe.h - hardware probes that bench.py times next to libtt's kernels (libttprobe.so).  NOT part of the product ABI of
 * include/tt.h and not linked into libtt.so: two self-contained kernels that measure what the roofline fractions are quoted
 * against on the GPU the bench runs on.  Same conventions as tt.h: 0 = success, negative = failure, `stream` is a cudaStream_t. */
#ifndef TT_PROBE_H_
#define TT_PROBE_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Read-only streaming probe: sums `bytes` (multiple of 16) of device memory at `src` with 128-bit loads that bypass L1 and
 * writes one 16-byte result per CTA to `sink` (>= 16*4096 bytes).  bench.py: the read-only HBM bandwidth next to the copy figure.
 * Returns -1 for a NULL pointer, -2 if bytes is not a multiple of 16, -9 for a CUDA launch error. */
int tt_probe_stream_read(const void* src, size_t bytes, void* sink, void* stream);

/* FP64 tensor-pipe probe: every warp of 148*8 CTAs x 256 threads issues iters x 16 independent mma.sync m8n8k4 f64 (DMMA);
 * *flops (host, may be NULL) receives the flop count of the launch.  sink: DEVICE, >= 148*8*256 doubles.  bench.py times it for
 * the measured DMMA peak the k-RHS roofline (configs[3]) is quoted against. */
int tt_probe_dmma(int iters, void* sink, double* flops, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* TT_PROBE_H_ */
