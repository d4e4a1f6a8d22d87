/* CPU ORACLE (test infrastructure, NOT the product path) - blocked/OpenMP build.
 *
 * Same sums as oracle/toeplitz_plain.py, i.e. the direct time-domain block
 * convolution that DEFINES the block lower-triangular Toeplitz p2o map
 * (eq 2.4-2.6), zero-based:
 *
 *     d_i[s]  = sum_{j<=i} sum_p F_{i-j}[s,p] m_j[p]                 (eq 2.5)
 *     m'_j[p] = sum_{i>=j} sum_s F_{i-j}[s,p] d_i[s]                 (its transpose,
 *                                                    PAPER.md:198, R2)
 *
 * with no FFT anywhere (the FFT algorithm of PAPER.md:265 is "exact up to
 * rounding error", so the definition is the oracle).  This
 * build only re-orders the loops so that it finishes on the larger configs
 * and can be timed as the CPU baseline: tiles over the space index p so the
 * working set stays in cache, OpenMP over independent outputs.  All products
 * and sums are fp64 (fp32 inputs are converted exactly).  Summation order is
 * fixed and independent of the thread count:
 *   matvec : for each output (i,s): p-tiles ascending; inside a tile j
 *            ascending; inside a (tile,j) dot product 8 interleaved partial
 *            sums (lane = p mod 8) combined pairwise at the end.
 *   rmatvec: for each output (j,p): i ascending, then s ascending.
 *
 * Layouts (time-major, the paper's stacking PAPER.md:83, 93-95), element
 * strides given explicitly so that sensor or parameter slices of the block
 * column can be passed without copying:
 *   F[k*ldk + s*lds + p]   block column F_k[s,p], k<N_t, s<N_d, p<N_m
 *   m[j*ldm + p], d[i*ldd + s]
 *
 * Shares no code with the CUDA path.  Pinned against toeplitz_plain.py and,
 * through it, against the pins listed there (tests/test_oracle_pins.py).
 */
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define TILE_P 1024

int tto_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

#define DEFINE_ORACLE(SUFFIX, T)                                                              \
/* 8-lane interleaved fp64 dot product of length n */                                         \
static double dot8_##SUFFIX(const T* a, const T* b, int64_t n) {                              \
    double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};                                                 \
    int64_t p = 0;                                                                            \
    for (; p + 8 <= n; p += 8)                                                                \
        for (int l = 0; l < 8; ++l) acc[l] += (double)a[p + l] * (double)b[p + l];            \
    for (int l = 0; p < n; ++p, ++l) acc[l] += (double)a[p] * (double)b[p];                   \
    return ((acc[0] + acc[1]) + (acc[2] + acc[3])) + ((acc[4] + acc[5]) + (acc[6] + acc[7])); \
}                                                                                             \
                                                                                              \
/* d[i*ldd + s] = sum_{j<=i} sum_p F_{i-j}[s,p] m_j[p]   for s in [0,N_d), i in [0,N_t) */     \
void tto_matvec_##SUFFIX(int64_t N_d, int64_t N_m, int64_t N_t, const T* F, int64_t ldk,      \
                         int64_t lds, const T* m, int64_t ldm, double* d, int64_t ldd) {      \
    for (int64_t i = 0; i < N_t; ++i)                                                         \
        for (int64_t s = 0; s < N_d; ++s) d[i * ldd + s] = 0.0;                               \
    for (int64_t p0 = 0; p0 < N_m; p0 += TILE_P) {                                            \
        int64_t np = N_m - p0 < TILE_P ? N_m - p0 : TILE_P;                                   \
        _Pragma("omp parallel for collapse(2) schedule(dynamic, 8)")                          \
        for (int64_t s = 0; s < N_d; ++s)                                                     \
            for (int64_t i = 0; i < N_t; ++i) {                                               \
                double acc = 0.0;                                                             \
                for (int64_t j = 0; j <= i; ++j)                                              \
                    acc += dot8_##SUFFIX(F + (i - j) * ldk + s * lds + p0, m + j * ldm + p0,  \
                                         np);                                                 \
                d[i * ldd + s] += acc;                                                        \
            }                                                                                 \
    }                                                                                         \
}                                                                                             \
                                                                                              \
/* out[j*ldo + p] = sum_{i>=j} sum_s F_{i-j}[s,p] d_i[s]   for p in [0,N_m), j in [0,N_t) */   \
void tto_rmatvec_##SUFFIX(int64_t N_d, int64_t N_m, int64_t N_t, const T* F, int64_t ldk,     \
                          int64_t lds, const T* d, int64_t ldd, double* out, int64_t ldo) {   \
    int64_t ntile = (N_m + TILE_P - 1) / TILE_P;                                              \
    _Pragma("omp parallel for collapse(2) schedule(dynamic, 4)")                              \
    for (int64_t t = 0; t < ntile; ++t)                                                       \
        for (int64_t j = 0; j < N_t; ++j) {                                                   \
            int64_t p0 = t * TILE_P;                                                          \
            int64_t np = N_m - p0 < TILE_P ? N_m - p0 : TILE_P;                               \
            double acc[TILE_P];                                                               \
            for (int64_t p = 0; p < np; ++p) acc[p] = 0.0;                                    \
            for (int64_t i = j; i < N_t; ++i)                                                 \
                for (int64_t s = 0; s < N_d; ++s) {                                           \
                    const T* row = F + (i - j) * ldk + s * lds + p0;                          \
                    double ds = (double)d[i * ldd + s];                                       \
                    for (int64_t p = 0; p < np; ++p) acc[p] += (double)row[p] * ds;           \
                }                                                                             \
            for (int64_t p = 0; p < np; ++p) out[j * ldo + p0 + p] = acc[p];                  \
        }                                                                                     \
}

DEFINE_ORACLE(f64, double)
DEFINE_ORACLE(f32, float)
