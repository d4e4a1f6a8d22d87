// tt_gemm32_umma.cu - the per-frequency complex64 GEMMs of TT_F32 plans with k right-hand sides on the 5th-generation tensor
// cores (step D of DESIGN.md for fp32; the many-matvec workloads of PAPER.md:296, 407, 421-423).  k a multiple of 16: 32 or 16
// columns per launch (template parameter kN = floats per row of the column group); the comments below are written for 32.
//
// forward   Dhat_w [N_d x k] = Fhat_w [N_d x N_m] * Xhat_w [N_m x k],  k = 32, as ONE real product per CTA tile
//
//     P [128 x 64] = A [128 x K] * B [K x 64],   K = parameters,
//     A rows   = 64 sensors x {Re Fhat_w[s, .], Im Fhat_w[s, .]}   (de-interleaved by the transform warps -> tensor memory)
//     B rows   = Xhat_w[p, .] exactly as it lies in memory: 32 complex = 64 floats (Re, Im interleaved), MN-major
//     Dhat_w[s, r] = (P[s.re, 2r] - P[s.im, 2r+1]) + i (P[s.re, 2r+1] + P[s.im, 2r])      (combined in the epilogue)
//
// so that all 128 x 64 accumulators carry useful terms and neither operand is transposed.  fp32 accuracy comes from the
// 3xTF32 split (x = hi + lo, both tf32; lo*hi + hi*lo + hi*hi, PAPER.md's fp32 runs need ~1e-6): Fhat is far too large
// to split ahead of time, so both operands are split on the fly by transform warps between TMA and the MMA:
//
//   warp 0      TMA producer: Fhat_w tile (64 sensors x 32 parameters, 16 KB) and Xhat_w tile (32 x 64 floats, 8 KB) per stage
//   warps 4-11  A transform: thread = tensor-memory lane = (sensor, re|im); reads its row from shared memory, splits, writes
//               hi and lo into tensor memory (tcgen05.st) - the MMA takes A from tensor memory, which halves the shared-memory
//               operand traffic that bounds small-N tcgen05 products.  Two warps per lane quadrant, alternating stages.
//   warps 2-3   B transform: element-wise hi / lo of the raw tile into two tiles in the MN-major operand layout
//   warp 1      tensor-memory allocation; MMA issuer: 4 k-steps x 3 tcgen05.mma (M 128, N 64, K 8) per stage
//   warps 12-15 epilogue: tensor-core fp32 accumulation truncates, so the accumulator is drained every kChunkKB stages
//               (two accumulators alternate) into fp32 register sums (round-to-nearest), as in tt_kdirect_umma.cu
//
// grid (p-splits, n_f, sensor tiles); the partial sums go through reduce_partials_kernel like those of the FMA kernel
// (tt_gemm32.cu), which stays the path for every other k and, for the adjoint, for N_d > 128.
#include "tt_common.cuh"
#include "tt_internal.h"
#include "tt_umma.cuh"

namespace tt {

namespace {

using namespace umma;

constexpr int kSens = 64;                      // sensors per CTA tile (128 tensor-memory lanes)
constexpr int kKB = 32;                        // parameters per pipeline stage
// (kN = floats per Xhat row handled by one launch = 2 x 32 or 2 x 16 columns is a template parameter of the kernels)
constexpr int kRaw = 6;                        // ring of raw tiles: filled by TMA, released by the transforms
constexpr int kOps = 4;                        // ring of operands (B hi / lo in shared, A hi / lo in tensor memory): -> MMA
constexpr int kChunkKB = 2;                    // stages per accumulation chunk (64 parameters)
constexpr int kRawA = kSens * kKB * 8;         // 16 KB: two TMA boxes of [64 rows][16 parameters = 128 B]
constexpr int kRawB = kKB * 64 * 4;            //  8 KB: raw [32 parameters][kN floats]; hi / lo [kN / 32 column halves][32][32 floats]
constexpr int kRawBytes = kRawA + kRawB, kOpBytes = 2 * kRawB;
constexpr int kFwdSmem = kRaw * kRawBytes + kOps * kOpBytes + 1024 /* alignment slack */ + 256 /* barriers */;
constexpr int kThreads = 512;
constexpr int kColD = 0;                       // two accumulators of 64 columns
constexpr int kColA = 128;                     // per stage: hi [32 columns], lo [32 columns]
constexpr int kTmemCols = 512;

__device__ __forceinline__ float4 lds128(uint32_t addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts128(uint32_t addr, uint4 v) {
    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

// x = hi + lo with hi = x rounded to tf32 (nearest, ties away: the bit pattern plus half a tf32 ulp, low 13 bits cleared -
// what cvt.rna.tf32.f32 computes, in two integer operations instead of the five the conversion expands to) and lo = the
// exact remainder.  lo is handed over with all its bits: the tensor core reads the upper 19 bits of a tf32 operand
// (measured: masking lo changes no bit of any result), and what it drops is below 2^-21 |x|, the size of the lo*lo term
// 3xTF32 leaves out anyway.
__device__ __forceinline__ void split_tf32(float x, uint32_t& hi, uint32_t& lo) {
    hi = (__float_as_uint(x) + 0x1000u) & 0xffffe000u;
    lo = __float_as_uint(x - __uint_as_float(hi));
}

// A raw stage may go back to the TMA producer only when the shared-memory loads from it have RETURNED.  An mbarrier arrive
// that merely follows the load instructions in program order does not wait for them (ptxas issues it under the loads'
// shadow; measured: tiles overwritten under the transform warps), so the arrive is made control-dependent on a warp
// vote over registers computed from the loaded values.  The vote is never true: a split hi part has 13 zero low bits.
__device__ __forceinline__ bool loads_returned(const uint32_t (&hi)[32]) {
    uint32_t f = hi[0];
#pragma unroll
    for (int j = 1; j < 32; ++j) f |= hi[j];
    return __ballot_sync(0xffffffffu, f == 0xffffffffu) == 0u;
}

template <int kN>
__global__ void __launch_bounds__(kThreads, 1)
gemm32_umma_fwd_kernel(const __grid_constant__ CUtensorMap mapF, const __grid_constant__ CUtensorMap mapX,
                       c64* __restrict__ partial, const GemmGeom g, const int r0) {
    extern __shared__ unsigned char smem_dyn[];
    const uint32_t smem0 = (smem_u32(smem_dyn) + 1023u) & ~1023u;
    const uint32_t ops0 = smem0 + kRaw * kRawBytes;
    const uint32_t bars = ops0 + kOps * kOpBytes;
    auto bar_full = [&](int s) { return bars + 8u * s; };                        // TMA -> transforms (raw tile landed)
    auto bar_rfree = [&](int s) { return bars + 8u * (kRaw + s); };              // transforms -> TMA (raw tile read)
    auto bar_ready = [&](int s) { return bars + 8u * (2 * kRaw + s); };          // transforms -> MMA (operands written)
    auto bar_free = [&](int s) { return bars + 8u * (2 * kRaw + kOps + s); };    // MMA -> transforms (operands consumed)
    auto bar_tfull = [&](int b) { return bars + 8u * (2 * kRaw + 2 * kOps + b); };   // MMA -> epilogue
    auto bar_tempty = [&](int b) { return bars + 8u * (2 * kRaw + 2 * kOps + 2 + b); };
    __shared__ uint32_t tmem_base_s;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int c = blockIdx.x, w = blockIdx.y, s0 = blockIdx.z * kSens;
    const long long p_lo = (long long)c * g.p_per_split;
    long long p_hi = p_lo + g.p_per_split;
    if (p_hi > g.N_m) p_hi = g.N_m;
    const int n_kb = p_hi > p_lo ? (int)((p_hi - p_lo + kKB - 1) / kKB) : 0;
    const int n_chunks = (n_kb + kChunkKB - 1) / kChunkKB;

    if (tid == 0) {
        for (int s = 0; s < kRaw; ++s) {
            mbar_init(bar_full(s), 1);
            mbar_init(bar_rfree(s), 6);   // 4 A-transform warps (one per lane quadrant) + 2 B-transform warps
        }
        for (int s = 0; s < kOps; ++s) {
            mbar_init(bar_ready(s), 6);
            mbar_init(bar_free(s), 1);
        }
        for (int b = 0; b < 2; ++b) {
            mbar_init(bar_tfull(b), 1);
            mbar_init(bar_tempty(b), 4);
        }
        mbar_fence_init();
        tma_prefetch_desc(&mapF);
        tma_prefetch_desc(&mapX);
    }
    if (warp == 1) tmem_alloc(smem_u32(&tmem_base_s), kTmemCols);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = tmem_base_s;

    if (warp == 0) {
        if (elect_one()) {
            for (int kb = 0; kb < n_kb; ++kb) {
                const int st = kb % kRaw;
                mbar_wait(bar_rfree(st), ((kb / kRaw) & 1) ^ 1);
                const uint32_t base = smem0 + st * kRawBytes;
                mbar_arrive_expect_tx(bar_full(st), kRawA + kKB * kN * 4);
                const long long p = p_lo + (long long)kb * kKB;
                tma_load_3d(base, &mapF, bar_full(st), (int)(2 * p), s0, w);
                tma_load_3d(base + kRawA / 2, &mapF, bar_full(st), (int)(2 * p + 32), s0, w);
                tma_load_3d(base + kRawA, &mapX, bar_full(st), 2 * r0, (int)p, w);
            }
        }
    } else if (warp == 1) {
        if (elect_one()) {
            constexpr uint32_t idesc = idesc_tf32(128, kN, /*b_mn_major=*/1);
            for (int kb = 0; kb < n_kb; ++kb) {
                const int st = kb % kOps, chunk = kb / kChunkKB, buf = chunk & 1;
                const bool first = kb % kChunkKB == 0;
                if (first) {
                    mbar_wait(bar_tempty(buf), ((chunk >> 1) & 1) ^ 1);
                    tc_fence_after();
                }
                mbar_wait(bar_ready(st), (kb / kOps) & 1);
                tc_fence_after();
                const uint32_t d = tmem_base + kColD + buf * 64;
                const uint32_t a_hi = tmem_base + kColA + st * 64, a_lo = a_hi + 32;
                const uint32_t b_hi = ops0 + st * kOpBytes, b_lo = b_hi + kRawB;
#pragma unroll
                for (int ks = 0; ks < kKB / 8; ++ks) {
                    const uint64_t dh = smem_desc_mnmajor_tf32(b_hi + ks * 1024, kKB * 128, 512);
                    const uint64_t dl = smem_desc_mnmajor_tf32(b_lo + ks * 1024, kKB * 128, 512);
                    mma_tf32_ts(d, a_lo + ks * 8, dh, idesc, (first && ks == 0) ? 0u : 1u);
                    mma_tf32_ts(d, a_hi + ks * 8, dl, idesc, 1u);
                    mma_tf32_ts(d, a_hi + ks * 8, dh, idesc, 1u);
                }
                tc_commit(bar_free(st));
                if (kb % kChunkKB == kChunkKB - 1 || kb == n_kb - 1) tc_commit(bar_tfull(buf));
            }
        }
    } else if (warp >= 4 && warp < 12) {
        // A transform: lane l of quadrant q is tensor-memory lane 32 q + l = sensor 16 q + (l & 15), part l >> 4; two warps
        // per quadrant take the stages in turn
        const int q = warp & 3, row = 16 * q + (lane & 15), part = lane >> 4;
        const uint32_t row_off = row * 128, sw = row & 7;
        for (int kb = (warp - 4) >> 2; kb < n_kb; kb += 2) {
            const int rs = kb % kRaw, st = kb % kOps;
            mbar_wait(bar_full(rs), (kb / kRaw) & 1);
            const uint32_t base = smem0 + rs * kRawBytes + row_off;
            uint32_t hi[32], lo[32];
#pragma unroll
            for (int b = 0; b < 2; ++b)
#pragma unroll
                for (int ch = 0; ch < 8; ++ch) {
                    const float4 v = lds128(base + b * (kRawA / 2) + ((ch ^ sw) << 4));
                    split_tf32(part ? v.y : v.x, hi[16 * b + 2 * ch], lo[16 * b + 2 * ch]);
                    split_tf32(part ? v.w : v.z, hi[16 * b + 2 * ch + 1], lo[16 * b + 2 * ch + 1]);
                }
            if (loads_returned(hi) && lane == 0) mbar_arrive(bar_rfree(rs));
            mbar_wait(bar_free(st), ((kb / kOps) & 1) ^ 1);
            tc_fence_after();
            const uint32_t ta = tmem_base + ((uint32_t)(32 * q) << 16) + kColA + st * 64;
            tmem_st_32x32(ta, hi);
            tmem_st_32x32(ta + 32, lo);
            tmem_st_wait();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_ready(st));
        }
    } else if (warp == 2 || warp == 3) {
        const int t = tid - 64;
        for (int kb = 0; kb < n_kb; ++kb) {
            const int rs = kb % kRaw, st = kb % kOps;
            mbar_wait(bar_full(rs), (kb / kRaw) & 1);
            // raw 16-byte piece t + 64 i = (row, c16) of the kN-float rows -> column half c16 / 8, row, piece c16 % 8 of the
            // operand layout, whose 32-byte pieces are XORed with row % 4
            constexpr int kPR = kN / 4, kPieces = kKB * kPR / 64, kRowStep = 64 / kPR;   // pieces per row, per thread; rows per pass
            const uint32_t raw = smem0 + rs * kRawBytes + kRawA + t * 16;
            const uint32_t c16 = t % kPR, row0 = t / kPR;
            float4 v[kPieces];
#pragma unroll
            for (int i = 0; i < kPieces; ++i) v[i] = lds128(raw + i * 1024);     // all loads in flight before the first use
            mbar_wait(bar_free(st), ((kb / kOps) & 1) ^ 1);
            const uint32_t dst0 = ops0 + st * kOpBytes + (c16 >> 3) * (kKB * 128) + row0 * 128 +
                                  ((((c16 & 7) >> 1) ^ (row0 & 3)) << 5) + ((c16 & 1) << 4);   // (row0 + kRowStep i) % 4 == row0 % 4
#pragma unroll
            for (int i = 0; i < kPieces; ++i) {
                uint4 h, l;
                split_tf32(v[i].x, h.x, l.x); split_tf32(v[i].y, h.y, l.y); split_tf32(v[i].z, h.z, l.z); split_tf32(v[i].w, h.w, l.w);
                sts128(dst0 + i * (kRowStep * 128), h);
                sts128(dst0 + i * (kRowStep * 128) + kRawB, l);
            }
            fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(bar_rfree(rs));
                mbar_arrive(bar_ready(st));
            }
        }
    } else if (warp >= 12) {
        const int q = warp & 3, part = lane >> 4;
        float acc[kN];
#pragma unroll
        for (int j = 0; j < kN; ++j) acc[j] = 0.f;
        for (int ch = 0; ch < n_chunks; ++ch) {
            const int buf = ch & 1;
            mbar_wait(bar_tfull(buf), (ch >> 1) & 1);
            tc_fence_after();
            const uint32_t ta = tmem_base + ((uint32_t)(32 * q) << 16) + kColD + buf * 64;
#pragma unroll
            for (int j = 0; j < kN / 16; ++j) {
                uint32_t v[16];
                tmem_ld_32x16(ta + 16 * j, v);
#pragma unroll
                for (int i = 0; i < 16; ++i) acc[16 * j + i] += __uint_as_float(v[i]);
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_tempty(buf));
        }
        // lanes l and l ^ 16 hold the Re-row and the Im-row products of one sensor: the Re lane finishes the first half of the
        // columns, the Im lane the second half
        constexpr int kH = kN / 2;                   // floats of half the columns
        float a[kH], b[kH];
#pragma unroll
        for (int j = 0; j < kH; ++j) {
            const float send = part ? acc[j] : acc[kH + j];
            const float recv = __shfl_xor_sync(0xffffffffu, send, 16);
            a[j] = part ? recv : acc[j];         // Re-row products of my columns
            b[j] = part ? acc[kH + j] : recv;    // Im-row products
        }
        const int s = s0 + 16 * q + (lane & 15);
        if (s < g.N_d) {
            float4* dst = reinterpret_cast<float4*>(partial + (((long long)w * g.split + c) * g.N_d + s) * g.k + r0 + (kH / 2) * part);
#pragma unroll
            for (int r = 0; r < kH / 2; r += 2)
                dst[r / 2] = make_float4(a[2 * r] - b[2 * r + 1], a[2 * r + 1] + b[2 * r], a[2 * r + 2] - b[2 * r + 3],
                                         a[2 * r + 3] + b[2 * r + 2]);
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc(tmem_base, kTmemCols);
}

// ---------------------------------------------------------------------------------------------------------------------
// adjoint   Xout_w [N_m x k] = Fhat_w^H [N_m x N_d] * Dhat_w [N_d x k],  k = 32, per tile of 128 parameters
//
//     P [128 x 64] = A [128 x K] * B [K x 64],   K = 2 N_d,
//     A[p, (s, 0)] = Re Fhat_w[s, p],  A[p, (s, 1)] = Im Fhat_w[s, p]      (thread p copies its (Re, Im) pairs: no shuffle)
//     B[(s, 0), .] = Dhat_w[s, .] as it lies in memory (Re, Im interleaved), B[(s, 1), .] = -i Dhat_w[s, .]
//     P[p, .]      = Xout_w[p, .] as it lies in memory
//
// B (hi and lo, the whole K) is built once per CTA and stays in shared memory: a CTA works through a range of parameter
// tiles of ONE frequency.  Per tile the Fhat_w tile streams through a TMA ring in K-blocks of 16 sensors (rows of 1 KB),
// the transform warps split it into tensor memory, and the MMA adds the hi*hi products into one accumulator and the two
// cross products into another (their sum is formed in the epilogue): the tensor core's truncating accumulation then acts
// once per k-step on the large terms instead of three times.  Tiles alternate between two accumulator pairs.
// ---------------------------------------------------------------------------------------------------------------------
constexpr int kAdjKB = 16;                         // sensors per K-block (32 K-columns)
constexpr int kAdjRawBytes = kAdjKB * 128 * 8;     // 16 KB: [16 sensors][128 parameters x 8 B]
constexpr int kAdjOps = 4;                         // tensor-memory ring of A operands
constexpr int kAdjColD = 0;                        // two accumulator pairs (hi*hi, cross) of 64 columns each
constexpr int kAdjColA = 256;
constexpr int kAdjSets = 2;                        // transform warps per lane quadrant
constexpr int kAdjThreads = 32 * (4 + 4 * kAdjSets + 4);   // TMA, MMA, 2 spare | transforms | 4 epilogue warps

struct AdjArgs {
    int n_raw;           // stages of the raw ring
    int n_kb;            // K-blocks per tile = ceil(N_d / 16)
    int tiles_per_cta;   // parameter tiles per CTA (grid.x CTAs per frequency)
    int n_tiles;         // ceil(N_m / 128)
};

template <int kN>
__global__ void __launch_bounds__(kAdjThreads, 1)
gemm32_umma_adj_kernel(const __grid_constant__ CUtensorMap mapF, const __grid_constant__ CUtensorMap mapX,
                       const c64* __restrict__ Dhat, const GemmGeom g, const AdjArgs a, const int r0) {
    extern __shared__ unsigned char smem_dyn[];
    const int krows = 2 * kAdjKB * a.n_kb;                              // K rows of B (padded sensors x 2)
    const uint32_t smem0 = (smem_u32(smem_dyn) + 1023u) & ~1023u;
    const uint32_t b_hi = smem0, b_lo = smem0 + krows * kN * 4;         // each: [kN / 32 column halves][krows][128 B]
    const uint32_t stg = smem0 + krows * kN * 8;                        // output tile: [kN / 32 column halves][128 rows][128 B]
    const uint32_t raw0 = stg + 128 * kN * 4;
    const uint32_t bars = raw0 + a.n_raw * kAdjRawBytes;
    constexpr int kMaxRaw = 12;
    auto bar_full = [&](int s) { return bars + 8u * s; };
    auto bar_rfree = [&](int s) { return bars + 8u * (kMaxRaw + s); };
    auto bar_ready = [&](int s) { return bars + 8u * (2 * kMaxRaw + s); };
    auto bar_free = [&](int s) { return bars + 8u * (2 * kMaxRaw + kAdjOps + s); };
    auto bar_tfull = [&](int b) { return bars + 8u * (2 * kMaxRaw + 2 * kAdjOps + b); };
    auto bar_tempty = [&](int b) { return bars + 8u * (2 * kMaxRaw + 2 * kAdjOps + 2 + b); };
    __shared__ uint32_t tmem_base_s;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int w = blockIdx.y;
    const int tile0 = blockIdx.x * a.tiles_per_cta;
    const int n_my = tile0 >= a.n_tiles ? 0 : (a.n_tiles - tile0 < a.tiles_per_cta ? a.n_tiles - tile0 : a.tiles_per_cta);
    const int n_it = n_my * a.n_kb;                                     // K-blocks this CTA streams

    if (tid == 0) {
        for (int s = 0; s < a.n_raw; ++s) {
            mbar_init(bar_full(s), 1);
            mbar_init(bar_rfree(s), 4);      // the 4 transform warps (one per lane quadrant) of the stage's set
        }
        for (int s = 0; s < kAdjOps; ++s) {
            mbar_init(bar_ready(s), 4);
            mbar_init(bar_free(s), 1);
        }
        for (int b = 0; b < 2; ++b) {
            mbar_init(bar_tfull(b), 1);
            mbar_init(bar_tempty(b), 4);
        }
        mbar_fence_init();
        tma_prefetch_desc(&mapF);
        tma_prefetch_desc(&mapX);
    }
    if (warp == 1) tmem_alloc(smem_u32(&tmem_base_s), kTmemCols);

    // B: 16-byte piece (s, c16) of Dhat_w = two complex columns -> rows 2 s and 2 s + 1, column half c16 / 8, piece c16 % 8
    {
        const c64* Dw = Dhat + (long long)w * g.N_d * g.k + r0;
        constexpr int kPR = kN / 4;                                      // 16-byte pieces per row of Dhat_w
        const int n_pieces = kAdjKB * a.n_kb * kPR;
        for (int idx = tid; idx < n_pieces; idx += kAdjThreads) {
            const int s = idx / kPR, c16 = idx % kPR;
            float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
            if (s < g.N_d) v = *reinterpret_cast<const float4*>(Dw + (long long)s * g.k + 2 * c16);
            const float4 u = make_float4(v.y, -v.x, v.w, -v.z);         // -i Dhat
            const uint32_t half = (uint32_t)(c16 >> 3) * (uint32_t)(krows * 128), sub = (uint32_t)(c16 & 1) << 4;
            const uint32_t p32 = (uint32_t)(c16 & 7) >> 1;
            const uint32_t k0 = 2 * s, k1 = 2 * s + 1;
            const uint32_t d0 = half + k0 * 128 + ((p32 ^ (k0 & 3)) << 5) + sub;
            const uint32_t d1 = half + k1 * 128 + ((p32 ^ (k1 & 3)) << 5) + sub;
            uint4 h, l;
            split_tf32(v.x, h.x, l.x); split_tf32(v.y, h.y, l.y); split_tf32(v.z, h.z, l.z); split_tf32(v.w, h.w, l.w);
            sts128(b_hi + d0, h);
            sts128(b_lo + d0, l);
            split_tf32(u.x, h.x, l.x); split_tf32(u.y, h.y, l.y); split_tf32(u.z, h.z, l.z); split_tf32(u.w, h.w, l.w);
            sts128(b_hi + d1, h);
            sts128(b_lo + d1, l);
        }
        fence_proxy_async_smem();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = tmem_base_s;

    if (warp == 0) {
        if (elect_one()) {
            int st = 0, ph = 0;
            for (int t = 0; t < n_my; ++t)
                for (int kb = 0; kb < a.n_kb; ++kb) {
                    mbar_wait(bar_rfree(st), ph ^ 1);
                    mbar_arrive_expect_tx(bar_full(st), kAdjRawBytes);
                    tma_load_3d(raw0 + st * kAdjRawBytes, &mapF, bar_full(st), (tile0 + t) * 256, kb * kAdjKB, w);
                    if (++st == a.n_raw) { st = 0; ph ^= 1; }
                }
        }
    } else if (warp == 1) {
        if (elect_one()) {
            constexpr uint32_t idesc = idesc_tf32(128, kN, /*b_mn_major=*/1);
            const uint32_t lbo = (uint32_t)krows * 128;
            int it = 0;
            for (int t = 0; t < n_my; ++t) {
                const int buf = t & 1;
                mbar_wait(bar_tempty(buf), ((t >> 1) & 1) ^ 1);
                tc_fence_after();
                const uint32_t d_h = tmem_base + kAdjColD + buf * 128, d_x = d_h + 64;
                for (int kb = 0; kb < a.n_kb; ++kb, ++it) {
                    const int st = it % kAdjOps;
                    mbar_wait(bar_ready(st), (it / kAdjOps) & 1);
                    tc_fence_after();
                    const uint32_t a_hi = tmem_base + kAdjColA + st * 64, a_lo = a_hi + 32;
#pragma unroll
                    for (int ks = 0; ks < 4; ++ks) {
                        const uint32_t off = (uint32_t)(kb * 32 + ks * 8) * 128;
                        const uint64_t dh = smem_desc_mnmajor_tf32(b_hi + off, lbo, 512);
                        const uint64_t dl = smem_desc_mnmajor_tf32(b_lo + off, lbo, 512);
                        const uint32_t acc = (kb > 0 || ks > 0) ? 1u : 0u;
                        mma_tf32_ts(d_x, a_lo + ks * 8, dh, idesc, acc);
                        mma_tf32_ts(d_x, a_hi + ks * 8, dl, idesc, 1u);
                        mma_tf32_ts(d_h, a_hi + ks * 8, dh, idesc, acc);
                    }
                    tc_commit(bar_free(st));
                }
                tc_commit(bar_tfull(buf));
            }
        }
    } else if (warp >= 4 && warp < 4 + 4 * kAdjSets) {
        // A transform: lane l of quadrant q is tensor-memory lane 32 q + l = parameter 32 q + l of the tile; column 2 j of the
        // stage = Re, 2 j + 1 = Im of sensor j of the K-block.  kAdjSets warps per quadrant take the K-blocks in turn.
        const int q = warp & 3, set = (warp - 4) >> 2;
        const uint32_t lane_off = (uint32_t)(32 * q + lane) * 8;
        int rs = set % a.n_raw, rph = (set / a.n_raw) & 1;              // raw stage and phase of K-block `it`
        for (int it = set; it < n_it; it += kAdjSets) {
            const int st = it % kAdjOps;
            mbar_wait(bar_full(rs), rph);
            const uint32_t base = raw0 + rs * kAdjRawBytes + lane_off;
            uint32_t hi[32], lo[32];
#pragma unroll
            for (int j = 0; j < kAdjKB; ++j) {
                float2 v;
                asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(base + j * 1024));
                split_tf32(v.x, hi[2 * j], lo[2 * j]);
                split_tf32(v.y, hi[2 * j + 1], lo[2 * j + 1]);
            }
            if (loads_returned(hi) && lane == 0) mbar_arrive(bar_rfree(rs));
            mbar_wait(bar_free(st), ((it / kAdjOps) & 1) ^ 1);
            tc_fence_after();
            const uint32_t ta = tmem_base + ((uint32_t)(32 * q) << 16) + kAdjColA + st * 64;
            tmem_st_32x32(ta, hi);
            tmem_st_32x32(ta + 32, lo);
            tmem_st_wait();
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_ready(st));
            rs += kAdjSets;
            while (rs >= a.n_raw) { rs -= a.n_raw; rph ^= 1; }
        }
    } else if (warp >= 4 + 4 * kAdjSets) {
        // epilogue: the tile leaves through shared memory and a TMA store.  (Each lane owns one 256-byte row of Xout_w: direct
        // stores put 16 bytes into each of 32 lines per instruction, and at 32 KB per tile that made the epilogue, not the
        // MMA, the pace of the kernel.)  Staging rows are 128 bytes per column half, 128-byte swizzled like the tensor map.
        const int q = warp & 3, row = 32 * q + lane;
        const bool leader = warp == 4 + 4 * kAdjSets && elect_one();
        const uint32_t srow = stg + (uint32_t)row * 128, sw = (uint32_t)row & 7;
        for (int t = 0; t < n_my; ++t) {
            const int buf = t & 1;
            mbar_wait(bar_tfull(buf), (t >> 1) & 1);
            tc_fence_after();
            if (leader) tma_store_wait_read();                          // the previous tile has left the staging buffer
            asm volatile("bar.sync 1, 128;" ::: "memory");
            const uint32_t ta = tmem_base + ((uint32_t)(32 * q) << 16) + kAdjColD + buf * 128;
#pragma unroll
            for (int j = 0; j < kN / 16; ++j) {
                uint32_t vh[16], vx[16];
                tmem_ld_32x16(ta + 16 * j, vh);
                tmem_ld_32x16(ta + 64 + 16 * j, vx);
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    uint4 o;
                    o.x = __float_as_uint(__uint_as_float(vh[4 * i]) + __uint_as_float(vx[4 * i]));
                    o.y = __float_as_uint(__uint_as_float(vh[4 * i + 1]) + __uint_as_float(vx[4 * i + 1]));
                    o.z = __float_as_uint(__uint_as_float(vh[4 * i + 2]) + __uint_as_float(vx[4 * i + 2]));
                    o.w = __float_as_uint(__uint_as_float(vh[4 * i + 3]) + __uint_as_float(vx[4 * i + 3]));
                    sts128(srow + (j >> 1) * (128 * 128) + ((((j & 1) * 4 + i) ^ sw) << 4), o);
                }
            }
            tc_fence_before();
            fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_tempty(buf));
            asm volatile("bar.sync 1, 128;" ::: "memory");
            if (leader) {
                tma_store_3d(&mapX, stg, 2 * r0, (tile0 + t) * 128, w);
                if (kN == 64) tma_store_3d(&mapX, stg + 128 * 128, 2 * r0 + 32, (tile0 + t) * 128, w);
                tma_store_commit();
            }
        }
        if (leader) tma_store_wait_all();
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc(tmem_base, kTmemCols);
}

int g_enable = 1;   // tt_debug_set("gemm32_umma", 0): keep to the FMA kernels

}  // namespace

void gemm32_umma_debug_set(int v) { g_enable = v; }

// The shapes the tensor-core path takes: groups of 32 columns (k a multiple of 32) or of 16 (k a multiple of 16).
bool gemm32_umma_fwd_ok(const GemmGeom& g) { return g_enable && g.k > 0 && g.k % 16 == 0 && 2 * g.ldp < (1LL << 31); }

cudaError_t gemm32_umma_fwd_launch(const void* Fhat, const void* Xhat, void* partial, const GemmGeom& g, cudaStream_t s) {
    const int n = g.k % 32 == 0 ? 64 : 32;       // floats per row handled by one launch
    CUtensorMap mapF, mapX;
    {   // Fhat as floats: [n_f][N_d][2 ldp]; box = 16 parameters x 64 sensors
        const unsigned long long dims[3] = {(unsigned long long)(2 * g.ldp), (unsigned long long)g.N_d, (unsigned long long)g.n_f};
        const unsigned long long strides[2] = {(unsigned long long)g.ldp * 8, (unsigned long long)g.N_d * g.ldp * 8};
        const unsigned box[3] = {32, kSens, 1};
        if (!make_tensor_map_f32(&mapF, Fhat, 3, dims, strides, box)) return cudaErrorInvalidValue;
    }
    {   // Xhat as floats: [n_f][N_m][2 k]; box = 64 floats x 32 parameters, rows as they lie in memory
        const unsigned long long dims[3] = {(unsigned long long)(2 * g.k), (unsigned long long)g.N_m, (unsigned long long)g.n_f};
        const unsigned long long strides[2] = {(unsigned long long)g.k * 8, (unsigned long long)g.ldx * 8};
        const unsigned box[3] = {(unsigned)n, kKB, 1};
        if (!make_tensor_map_f32(&mapX, Xhat, 3, dims, strides, box, /*swizzle128=*/false)) return cudaErrorInvalidValue;
    }
    auto kern = n == 64 ? gemm32_umma_fwd_kernel<64> : gemm32_umma_fwd_kernel<32>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kFwdSmem);
    if (e != cudaSuccess) return e;
    const dim3 grid((unsigned)g.split, (unsigned)g.n_f, (unsigned)((g.N_d + kSens - 1) / kSens));
    for (int r0 = 0; r0 < g.k; r0 += n / 2) {
        kern<<<grid, kThreads, kFwdSmem, s>>>(mapF, mapX, static_cast<c64*>(partial), g, r0);
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

// adjoint: the whole K (2 N_d rows of B, hi and lo) stays in shared memory beside a raw ring of at least 4 stages
bool gemm32_umma_adj_ok(const GemmGeom& g) {
    return g_enable && g.k > 0 && g.k % 16 == 0 && g.N_d <= 128 && 2 * g.ldp < (1LL << 31);
}

cudaError_t gemm32_umma_adj_launch(const void* Fhat, const void* Dhat, void* Xhat_out, const GemmGeom& g, cudaStream_t s) {
    const int n = g.k % 32 == 0 ? 64 : 32;       // floats per row handled by one launch
    CUtensorMap mapF;
    {   // Fhat as floats: [n_f][N_d][2 ldp]; box = 128 parameters (1 KB) x 16 sensors, no swizzle (thread p reads 8 B at 8 p)
        const unsigned long long dims[3] = {(unsigned long long)(2 * g.ldp), (unsigned long long)g.N_d, (unsigned long long)g.n_f};
        const unsigned long long strides[2] = {(unsigned long long)g.ldp * 8, (unsigned long long)g.N_d * g.ldp * 8};
        const unsigned box[3] = {256, kAdjKB, 1};
        if (!make_tensor_map_f32(&mapF, Fhat, 3, dims, strides, box, /*swizzle128=*/false)) return cudaErrorInvalidValue;
    }
    CUtensorMap mapX;
    {   // Xout as floats: [n_f][N_m][2 k]; box = 32 floats (one column half) x 128 parameters, 128-byte swizzle
        const unsigned long long dims[3] = {(unsigned long long)(2 * g.k), (unsigned long long)g.N_m, (unsigned long long)g.n_f};
        const unsigned long long strides[2] = {(unsigned long long)g.k * 8, (unsigned long long)g.ldx * 8};
        const unsigned box[3] = {32, 128, 1};
        if (!make_tensor_map_f32(&mapX, Xhat_out, 3, dims, strides, box)) return cudaErrorInvalidValue;
    }
    AdjArgs a;
    a.n_kb = (g.N_d + kAdjKB - 1) / kAdjKB;
    a.n_tiles = (int)((g.N_m + 127) / 128);
    const int b_bytes = 2 * kAdjKB * a.n_kb * n * 8, stg_bytes = 128 * n * 4;
    a.n_raw = (232448 - 2048 - b_bytes - stg_bytes) / kAdjRawBytes;
    if (a.n_raw > 12) a.n_raw = 12;
    // Every raw stage must belong to ONE set of transform warps.  A set meets its stages in order, so it cannot reach a
    // stage a whole phase early; a second set could, and a parity wait cannot tell "the phase before last has completed"
    // from "the phase I am waiting for has completed" (measured with 5 stages and 2 sets: tiles read before they landed).
    a.n_raw -= a.n_raw % kAdjSets;
    if (a.n_raw < 4) return cudaErrorInvalidValue;
    const int smem = b_bytes + stg_bytes + a.n_raw * kAdjRawBytes + 1024 + 512;
    // CTAs per frequency: ~6 waves over the SMs, at least 8 tiles each so that building B stays a small part
    int dev = 0, sms = 148;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    int per_f = (6 * sms + g.n_f - 1) / g.n_f;
    if (per_f > (a.n_tiles + 7) / 8) per_f = (a.n_tiles + 7) / 8;
    if (per_f < 1) per_f = 1;
    a.tiles_per_cta = (a.n_tiles + per_f - 1) / per_f;
    per_f = (a.n_tiles + a.tiles_per_cta - 1) / a.tiles_per_cta;
    auto kern = n == 64 ? gemm32_umma_adj_kernel<64> : gemm32_umma_adj_kernel<32>;
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    const dim3 grid((unsigned)per_f, (unsigned)g.n_f);
    for (int r0 = 0; r0 < g.k; r0 += n / 2) {
        kern<<<grid, kAdjThreads, smem, s>>>(mapF, mapX, static_cast<const c64*>(Dhat), g, a, r0);
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

}  // namespace tt
