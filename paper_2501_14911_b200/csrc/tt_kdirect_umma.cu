// tt_kdirect_umma.cu - C (+)= A B^T for fp32 row-major A (nA x Kdim), B (nB x Kdim) on the 5th-generation tensor cores:
// the one real GEMM  W = Fcol Gcol^T  of tt_assemble_K_direct (and the rectangular products of tt_qoi_direct), a dense
// contraction of n^2 N_m multiply-adds (7.9e13 for the lower triangle at the paper's shape).
//
// fp32 accuracy from tf32 tensor cores (the 1e-5 bar of K is relative to |K|_F; a plain tf32 product has 2^-11 per factor):
// every factor is split  a = hi + lo,  hi = tf32(a) (round to nearest), lo = tf32(a - hi)  (a - hi is exact in fp32), and
//     a b  ~=  hi_a hi_b + hi_a lo_b + lo_a hi_b            (the dropped lo_a lo_b and the rounding of lo are <= 2^-21 |a b|)
// is three tcgen05.mma kind::tf32 per k-step into the same fp32 accumulator in tensor memory.
//
//   kd_split_kernel   one pass over a slab of `ks` parameters of A and B: hi and lo parts, written K-major with an aligned
//                     pitch (the block columns themselves have no alignment: N_m = 263 169 is odd), zero-filled to a
//                     multiple of the K-block.  HBM-bound, 6 x the slab's bytes.
//   kd_umma_kernel    persistent, warp-specialised, one CTA of 12 warps per SM.  Tile 128 x 256 of C per step:
//                       warp 0   TMA producer: cp.async.bulk.tensor of the four operand tiles (A hi, A lo, B hi, B lo;
//                                128-byte swizzle, K-major) into a ring of shared-memory stages, mbarrier complete_tx
//                       warp 1   MMA issuer: one thread, tcgen05.mma cta_group::1 kind::tf32 M = 128, N = 256, K = 8,
//                                3 products x (K-block / 8) per stage; tcgen05.commit frees the stage and, every 128
//                                parameters (a CHUNK), publishes the accumulator
//                       warp 2   allocates the 512 columns of tensor memory: two 128 x 256 fp32 accumulators used in
//                                turn, so the epilogue of chunk c runs under the MMAs of chunk c + 1
//                       warps 4-11  epilogue (two warpgroups, setmaxnreg 232): tcgen05.ld of the finished chunk (32 lanes
//                                x 16 columns per instruction), fp32 running sums in registers (128 per thread); at the end
//                                of a tile C[row][col] (+)= (double) sum
//                     Why chunks: the tensor core adds each K = 8 product into its fp32 accumulator with truncation; the
//                     relative error of C measured 1.1e-8 x (parameters accumulated in tensor memory): 4.5e-5 after 4096.
//                     With 128-parameter chunks summed in registers with round-to-nearest it is 1.1e-6 at any length.
//                     Slab sums meet in fp64 in C in a fixed order (slab after slab on one stream): bit-reproducible.
#include <cuda.h>

#include <mutex>
#include <new>

#include "../../include/tt.h"
#include "tt_common.cuh"
#include "tt_internal.h"
#include "tt_umma.cuh"

// Scratch of kd_umma_gemm_static (the entry point tt_assemble_K_direct_static, which may not allocate): a fixed 64 MiB of
// device memory that every GPU loading this library holds until the process exits.  In HOST code this name is only a
// stand-in for the symbol - the device address comes from cudaGetSymbolAddress, once per device (static_scratch() below).
constexpr size_t kStaticScratchBytes = (size_t)64 << 20;
static __device__ __align__(256) unsigned char g_kd_static_scratch[kStaticScratchBytes];

namespace tt {
namespace {

using namespace umma;

constexpr int kBM = 128, kBN = 256;                 // C tile
// K-block BK = floats of K per shared-memory stage and operand row = one swizzle span: 32 (128-byte swizzle, 96 KB per stage,
// two stages).  BK = 16 (64-byte swizzle, four stages of 48 KB) was measured slower at the paper's shape: 1.09 s against 0.80 - 0.91 s.
template <int BK> struct Geo {
    static constexpr int kStages = BK == 32 ? 2 : 4;
    static constexpr int kABytes = kBM * BK * 4, kBBytes = kBN * BK * 4;
    static constexpr int kStageBytes = 2 * kABytes + 2 * kBBytes;   // A hi, A lo, B hi, B lo
    static constexpr int kChunkBlocks = 128 / BK;   // K-blocks accumulated in tensor memory between register flushes (128 parameters)
    static constexpr int kSmemBytes = kStages * kStageBytes + 1024 /* alignment slack */ + 256 /* barriers, tmem address */;
};
constexpr int kMaxBK = 32;                          // slabs are padded to a multiple of this
constexpr int kCtrlWarps = 4, kEpiWarps = 8;        // warpgroup 0: TMA / MMA / tensor-memory allocation; warpgroups 1-2: epilogue
constexpr int kThreads = 32 * (kCtrlWarps + kEpiWarps);
constexpr int kAccCols = kBN;                       // fp32 accumulator: one tensor-memory column per C column
constexpr int kPanel = 8;                           // tile columns per panel of the tile order

// hi / lo split of one slab: dst_hi/dst_lo[row][0..kpad) for src[row][k0 .. k0 + ks), zero beyond ks (kpad = ks rounded
// up to the K-block).  One warp per (row, 1024-parameter segment); a lane owns four consecutive parameters: four scalar
// loads (the rows of a block column have no alignment; the warp's four load instructions share their cache lines) and one
// 16-byte store per output (the scratch rows are 128-byte aligned).
__global__ void __launch_bounds__(256)
kd_split_kernel(const float* __restrict__ src, const long long rows, const long long ld, const long long k0, const int ks,
                const int kpad, float* __restrict__ dst_hi, float* __restrict__ dst_lo, const long long pitch) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long row = (long long)blockIdx.x * 8 + warp;
    if (row >= rows) return;
    const float* s = src + row * ld + k0;
    float* h = dst_hi + row * pitch;
    float* l = dst_lo + row * pitch;
    const int seg0 = blockIdx.y * 1024;
#pragma unroll 2
    for (int i = 0; i < 8; ++i) {
        const int k = seg0 + i * 128 + lane * 4;
        if (k >= kpad) break;                      // kpad is a multiple of 32: a lane's four parameters are in or out together
        float a[4], hi[4], lo[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) a[j] = k + j < ks ? __ldg(s + k + j) : 0.f;
#pragma unroll
        for (int j = 0; j < 4; ++j) { hi[j] = to_tf32(a[j]); lo[j] = to_tf32(a[j] - hi[j]); }
        *reinterpret_cast<float4*>(h + k) = make_float4(hi[0], hi[1], hi[2], hi[3]);
        *reinterpret_cast<float4*>(l + k) = make_float4(lo[0], lo[1], lo[2], lo[3]);
    }
}

// The C tiles to compute, in the order the persistent CTAs take them (CTA b takes entries b, b + grid, ...): panels of kPanel
// tile columns, inside a panel row by row.  The ~148 tiles in flight at any time are then ~18 tile rows x 8 tile columns that
// walk through K together, so a K-block of A or B fetched from HBM is served to 8 / 18 CTAs from L2.  lower_only: only the
// tiles that touch the lower triangle (tile row tm has (tm + 2) / 2 of them: 128-row tiles against 256-column tiles).
__host__ __device__ inline long long kd_tile_order(int2* out, int tm_n, int tn_n, int lower_only) {
    long long n = 0;
    for (int p0 = 0; p0 < tn_n; p0 += kPanel)
        for (int tm = lower_only ? (2 * p0 > 0 ? 2 * p0 - 1 : 0) : 0; tm < tm_n; ++tm) {
            int hi = p0 + kPanel < tn_n ? p0 + kPanel : tn_n;
            if (lower_only && (tm + 2) / 2 < hi) hi = (tm + 2) / 2;
            for (int tn = p0; tn < hi; ++tn, ++n)
                if (out) out[n] = make_int2(tm, tn);
        }
    return n;
}
__global__ void kd_tiles_kernel(int2* out, int tm_n, int tn_n, int lower_only) {
    if (blockIdx.x == 0 && threadIdx.x == 0) kd_tile_order(out, tm_n, tn_n, lower_only);
}

// (double)x as a volatile statement: the compiler otherwise converts all 128 running sums of a thread up front and spills
__device__ __forceinline__ double to_f64_here(float x) {
    double d;
    asm volatile("cvt.f64.f32 %0, %1;" : "=d"(d) : "f"(x));
    return d;
}

struct UmmaArgs {
    const int2* tiles;     // (tm, tn) of the C tiles, in processing order
    int n_tiles;
    int n_kblocks;         // K-blocks of this slab
    double* C;
    long long nA, nB, ldc;
    int first;             // 1: C = acc (first slab), 0: C += acc
};

template <int BK>
__global__ void __launch_bounds__(kThreads, 1)
kd_umma_kernel(const __grid_constant__ CUtensorMap tmA_hi, const __grid_constant__ CUtensorMap tmA_lo,
               const __grid_constant__ CUtensorMap tmB_hi, const __grid_constant__ CUtensorMap tmB_lo, const UmmaArgs g) {
    constexpr int kBK = BK, kStages = Geo<BK>::kStages, kABytes = Geo<BK>::kABytes, kBBytes = Geo<BK>::kBBytes,
                  kStageBytes = Geo<BK>::kStageBytes, kChunkBlocks = Geo<BK>::kChunkBlocks;
    extern __shared__ unsigned char smem_raw[];
    const uint32_t base = (smem_u32(smem_raw) + 1023u) & ~1023u;       // swizzle atoms want 1024-byte alignment
    const uint32_t bars = base + kStages * kStageBytes;                // full[S], empty[S], tmem_full[2], tmem_empty[2]
    auto full_bar = [&](int s) { return bars + 8u * s; };
    auto empty_bar = [&](int s) { return bars + 8u * (kStages + s); };
    auto tfull_bar = [&](int b) { return bars + 8u * (2 * kStages + b); };
    auto tempty_bar = [&](int b) { return bars + 8u * (2 * kStages + 2 + b); };
    const uint32_t tmem_slot = bars + 8u * (2 * kStages + 4);
    volatile uint32_t* tmem_slot_ptr =
        reinterpret_cast<volatile uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (warp == 0 && lane == 0) {
        tma_prefetch_desc(&tmA_hi); tma_prefetch_desc(&tmA_lo); tma_prefetch_desc(&tmB_hi); tma_prefetch_desc(&tmB_lo);
    }
    if (warp == 1 && lane == 0) {
        for (int s = 0; s < kStages; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
        for (int b = 0; b < 2; ++b) { mbar_init(tfull_bar(b), 1); mbar_init(tempty_bar(b), kEpiWarps); }
        mbar_fence_init();
    }
    if (warp == 2) tmem_alloc(tmem_slot, 2 * kAccCols);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;
    const int n_chunks = (g.n_kblocks + kChunkBlocks - 1) / kChunkBlocks;   // per tile

    if (warp < kCtrlWarps) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 32;");           // hand the registers to the epilogue warpgroups
        if (warp == 0 && elect_one()) {
            // ===== TMA producer =====
            int stage = 0;
            uint32_t phase = 0;
            for (int t = blockIdx.x; t < g.n_tiles; t += gridDim.x) {
                const int2 tile = g.tiles[t];
                const int rowA = tile.x * kBM, rowB = tile.y * kBN;
                for (int kb = 0; kb < g.n_kblocks; ++kb) {
                    mbar_wait(empty_bar(stage), phase ^ 1u);
                    const uint32_t sa = base + stage * kStageBytes;
                    mbar_arrive_expect_tx(full_bar(stage), kStageBytes);
                    tma_load_2d(sa, &tmA_hi, full_bar(stage), kb * kBK, rowA);
                    tma_load_2d(sa + kABytes, &tmA_lo, full_bar(stage), kb * kBK, rowA);
                    tma_load_2d(sa + 2 * kABytes, &tmB_hi, full_bar(stage), kb * kBK, rowB);
                    tma_load_2d(sa + 2 * kABytes + kBBytes, &tmB_lo, full_bar(stage), kb * kBK, rowB);
                    if (++stage == kStages) { stage = 0; phase ^= 1u; }
                }
            }
        } else if (warp == 1 && elect_one()) {
            // ===== MMA issuer: one chunk of kChunkBlocks K-blocks per tensor-memory accumulator, the two accumulators in turn =====
            constexpr uint32_t idesc = idesc_tf32(kBM, kBN);
            int stage = 0;
            uint32_t phase = 0;
            uint32_t cc = 0;                                            // chunks issued so far
            for (int t = blockIdx.x; t < g.n_tiles; t += gridDim.x) {
                for (int kb0 = 0; kb0 < g.n_kblocks; kb0 += kChunkBlocks, ++cc) {
                    const uint32_t buf = cc & 1u;
                    mbar_wait(tempty_bar(buf), ((cc >> 1) & 1u) ^ 1u);  // the epilogue has drained this accumulator
                    tc_fence_after();
                    const uint32_t d = tmem_base + buf * kAccCols;
                    const int kb1 = kb0 + kChunkBlocks < g.n_kblocks ? kb0 + kChunkBlocks : g.n_kblocks;
                    for (int kb = kb0; kb < kb1; ++kb) {
                        mbar_wait(full_bar(stage), phase);              // the four tiles of this stage have landed
                        tc_fence_after();
                        const uint32_t sa = base + stage * kStageBytes;
                        const uint64_t a_hi = smem_desc_kmajor<4 * BK>(sa), a_lo = smem_desc_kmajor<4 * BK>(sa + kABytes);
                        const uint64_t b_hi = smem_desc_kmajor<4 * BK>(sa + 2 * kABytes),
                                       b_lo = smem_desc_kmajor<4 * BK>(sa + 2 * kABytes + kBBytes);
#pragma unroll
                        for (int k = 0; k < kBK / 8; ++k) {             // 8 tf32 = 32 bytes along K: + 2 in the address field
                            const uint64_t o = (uint64_t)(k * 2);
                            mma_tf32(d, a_lo + o, b_hi + o, idesc, (kb > kb0 || k > 0) ? 1u : 0u);
                            mma_tf32(d, a_hi + o, b_lo + o, idesc, 1u);
                            mma_tf32(d, a_hi + o, b_hi + o, idesc, 1u);
                        }
                        tc_commit(empty_bar(stage));                    // stage free once these MMAs have read it
                        if (++stage == kStages) { stage = 0; phase ^= 1u; }
                    }
                    tc_commit(tfull_bar(buf));                          // chunk complete
                }
            }
        }
    } else {
        // ===== epilogue: per chunk tensor memory -> fp32 running sums in registers; per tile registers -> C (fp64) =====
        // The tensor core adds every K = 8 product into the fp32 accumulator with truncation (measured: a relative bias of
        // ~1e-8 per accumulated parameter), so accumulators are kept short (one chunk) and the chunk sums are added here
        // with round-to-nearest.
        asm volatile("setmaxnreg.inc.sync.aligned.u32 232;");
        const int q = warp & 3;                                         // this warp's 32 lanes of tensor memory (rows of the tile)
        const int h = (warp - kCtrlWarps) >> 2;                         // column half of the tile
        float acc[kBN / 2];
#pragma unroll
        for (int j = 0; j < kBN / 2; ++j) acc[j] = 0.f;
        uint32_t cc = 0;
        for (int t = blockIdx.x; t < g.n_tiles; t += gridDim.x) {
            for (int c = 0; c < n_chunks; ++c, ++cc) {
                const uint32_t buf = cc & 1u;
                mbar_wait(tfull_bar(buf), (cc >> 1) & 1u);
                tc_fence_after();
                const uint32_t ta = tmem_base + ((uint32_t)(q * 32) << 16) + buf * kAccCols + (uint32_t)(h * (kBN / 2));
#pragma unroll
                for (int c16 = 0; c16 < kBN / 2; c16 += 16) {
                    uint32_t r[16];
                    tmem_ld_32x16(ta + (uint32_t)c16, r);
#pragma unroll
                    for (int j = 0; j < 16; ++j) acc[c16 + j] += __uint_as_float(r[j]);
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(tempty_bar(buf));
            }
            const int2 tile = g.tiles[t];
            const long long row = (long long)tile.x * kBM + q * 32 + lane;
            const long long col0 = (long long)tile.y * kBN + h * (kBN / 2);
            double* crow = g.C + row * g.ldc + col0;
            if (row < g.nA) {
#pragma unroll
                for (int j0 = 0; j0 < kBN / 2; j0 += 8) {              // 8 doubles = 64 contiguous bytes at a time
                    double v[8];
#pragma unroll
                    for (int j = 0; j < 8; ++j) v[j] = (g.first || col0 + j0 + j >= g.nB) ? 0.0 : crow[j0 + j];
#pragma unroll
                    for (int j = 0; j < 8; ++j)
                        if (col0 + j0 + j < g.nB) crow[j0 + j] = v[j] + to_f64_here(acc[j0 + j]);
                    asm volatile("" ::: "memory");                      // keep the groups apart: registers
                }
            }
#pragma unroll
            for (int j = 0; j < kBN / 2; ++j) acc[j] = 0.f;
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 2) tmem_dealloc(tmem_base, 2 * kAccCols);
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

// rows x kpad floats, row pitch `pitch` floats (a multiple of 4), boxes of box_rows x 32 floats, 128-byte swizzle; rows
// beyond `rows` read as zeros
bool make_map(CUtensorMap* m, float* ptr, long long rows, int kpad, long long pitch, int box_rows, int bk) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return false;
    const cuuint64_t gdim[2] = {(cuuint64_t)kpad, (cuuint64_t)rows};
    const cuuint64_t gstride[1] = {(cuuint64_t)pitch * 4};
    const cuuint32_t box[2] = {(cuuint32_t)bk, (cuuint32_t)box_rows};
    const cuuint32_t estr[2] = {1, 1};
    return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, ptr, gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
              bk == 32 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

int g_slab = 0;   // tt_debug_set("kd_slab"): parameters per slab (0 = default)

}  // namespace

void kd_umma_debug_set_slab(int ks) { g_slab = ks; }

// C (nA x nB, fp64, pitch ldc) = A B^T, A: nA x Kdim, B: nB x Kdim, fp32 row-major with pitch Kdim (any alignment);
// lower_only: only the tiles that touch the lower triangle (nA == nB).  Stream-ordered: scratch comes from
// cudaMallocAsync / cudaFreeAsync on `s`, nothing synchronises.
cudaError_t kd_umma_gemm(const float* A, const float* B, double* C, long long nA, long long nB, long long Kdim, long long ldc,
                         int lower_only, cudaStream_t s) {
    // slab: parameters per pass of the split + GEMM pair; its sums meet the earlier slabs' in fp64 in C
    long long ks_max = g_slab > 0 ? g_slab : 8192;
    constexpr int bk = 32;
    ks_max = (ks_max + kMaxBK - 1) / kMaxBK * kMaxBK;
    if (ks_max > Kdim) ks_max = (Kdim + kMaxBK - 1) / kMaxBK * kMaxBK;
    const long long pitch = ks_max;                                     // floats; a multiple of 32
    const int tm_n = (int)((nA + kBM - 1) / kBM), tn_n = (int)((nB + kBN - 1) / kBN);
    const long long n_tiles_ll = kd_tile_order(nullptr, tm_n, tn_n, lower_only);
    if (n_tiles_ll > 0x7fffffffLL) return cudaErrorInvalidValue;
    const int n_tiles = (int)n_tiles_ll;

    float* scratch = nullptr;
    int2* d_tiles = nullptr;
    const size_t plane_a = (size_t)nA * pitch, plane_b = (size_t)nB * pitch;
    cudaError_t e = cudaMallocAsync(reinterpret_cast<void**>(&scratch), (2 * plane_a + 2 * plane_b) * sizeof(float), s);
    if (e != cudaSuccess) return e;
    e = cudaMallocAsync(reinterpret_cast<void**>(&d_tiles), (size_t)n_tiles * sizeof(int2), s);
    if (e != cudaSuccess) { cudaFreeAsync(scratch, s); return e; }
    kd_tiles_kernel<<<1, 32, 0, s>>>(d_tiles, tm_n, tn_n, lower_only);
    float *a_hi = scratch, *a_lo = scratch + plane_a, *b_hi = scratch + 2 * plane_a, *b_lo = b_hi + plane_b;

    CUtensorMap mA_hi, mA_lo, mB_hi, mB_lo;
    if (!(make_map(&mA_hi, a_hi, nA, (int)ks_max, pitch, kBM, bk) && make_map(&mA_lo, a_lo, nA, (int)ks_max, pitch, kBM, bk) &&
          make_map(&mB_hi, b_hi, nB, (int)ks_max, pitch, kBN, bk) && make_map(&mB_lo, b_lo, nB, (int)ks_max, pitch, kBN, bk)))
        e = cudaErrorInvalidValue;
    constexpr int smem = Geo<bk>::kSmemBytes;
    if (e == cudaSuccess) e = cudaFuncSetAttribute(kd_umma_kernel<bk>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    int dev = 0, sms = 148;
    if (e == cudaSuccess) e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int grid = n_tiles < sms ? n_tiles : sms;
    for (long long k0 = 0; e == cudaSuccess && k0 < Kdim; k0 += ks_max) {
        const int ks = (int)(Kdim - k0 < ks_max ? Kdim - k0 : ks_max);
        const int kpad = (ks + kMaxBK - 1) / kMaxBK * kMaxBK;
        const dim3 ga((unsigned)((nA + 7) / 8), (unsigned)((kpad + 1023) / 1024)), gb((unsigned)((nB + 7) / 8), ga.y);
        kd_split_kernel<<<ga, 256, 0, s>>>(A, nA, Kdim, k0, ks, kpad, a_hi, a_lo, pitch);
        kd_split_kernel<<<gb, 256, 0, s>>>(B, nB, Kdim, k0, ks, kpad, b_hi, b_lo, pitch);
        UmmaArgs g{d_tiles, n_tiles, kpad / bk, C, nA, nB, ldc, k0 == 0 ? 1 : 0};
        kd_umma_kernel<bk><<<grid, kThreads, smem, s>>>(mA_hi, mA_lo, mB_hi, mB_lo, g);
        e = cudaGetLastError();
    }
    cudaFreeAsync(d_tiles, s);
    cudaFreeAsync(scratch, s);
    return e;
}

namespace {

constexpr int kMaxDevices = 64;

// Device address of g_kd_static_scratch on the CURRENT device; looked up once per device, with that device current.
cudaError_t static_scratch(unsigned char** out) {
    static std::mutex mu;
    static unsigned char* ptrs[kMaxDevices] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (!ptrs[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_kd_static_scratch);
        if (e != cudaSuccess) return e;
        ptrs[dev] = static_cast<unsigned char*>(p);
    }
    *out = ptrs[dev];
    return cudaSuccess;
}

}  // namespace

// kd_umma_gemm with its scratch (hi / lo planes of one slab of A and B, the tile list) in g_kd_static_scratch instead of the
// stream-ordered allocator: no cudaMalloc* / cudaFree* of any kind.  The slab shrinks until the planes fit (at least 128
// parameters, or all of them); *fits = 0 and nothing is launched when even that does not fit.  Nothing in the scratch has to
// start at zero: every slab pass rewrites the part of the planes it reads (the split kernel zero-fills up to the K-block) and
// the tile list is rebuilt per call.  All calls on a device share the array: calls that overlap on the GPU race.
cudaError_t kd_umma_gemm_static(const float* A, const float* B, double* C, long long nA, long long nB, long long Kdim,
                                long long ldc, int lower_only, cudaStream_t s, int* fits) {
    *fits = 0;
    constexpr int bk = 32;
    const int tm_n = (int)((nA + kBM - 1) / kBM), tn_n = (int)((nB + kBN - 1) / kBN);
    const long long n_tiles_ll = kd_tile_order(nullptr, tm_n, tn_n, lower_only);
    if (n_tiles_ll > 0x7fffffffLL) return cudaSuccess;
    const int n_tiles = (int)n_tiles_ll;
    const long long kfull = (Kdim + kMaxBK - 1) / kMaxBK * kMaxBK;
    const long long tiles_bytes = ((long long)n_tiles * (long long)sizeof(int2) + 255) / 256 * 256;
    const long long row_bytes = 4 * (2 * nA + 2 * nB);                     // bytes of the four planes per parameter
    long long ks_max = ((long long)kStaticScratchBytes - tiles_bytes) / row_bytes / kMaxBK * kMaxBK;
    if (ks_max > 8192) ks_max = 8192;
    if (ks_max > kfull) ks_max = kfull;
    if (ks_max < (kfull < 128 ? kfull : 128)) return cudaSuccess;          // does not fit
    *fits = 1;

    unsigned char* base = nullptr;
    cudaError_t e = static_scratch(&base);
    if (e != cudaSuccess) return e;
    const long long pitch = ks_max;
    const size_t plane_a = (size_t)nA * pitch, plane_b = (size_t)nB * pitch;
    float* a_hi = reinterpret_cast<float*>(base);
    float *a_lo = a_hi + plane_a, *b_hi = a_hi + 2 * plane_a, *b_lo = b_hi + plane_b;
    int2* d_tiles = reinterpret_cast<int2*>(base + kStaticScratchBytes - tiles_bytes);
    kd_tiles_kernel<<<1, 32, 0, s>>>(d_tiles, tm_n, tn_n, lower_only);

    CUtensorMap mA_hi, mA_lo, mB_hi, mB_lo;
    if (!(make_map(&mA_hi, a_hi, nA, (int)ks_max, pitch, kBM, bk) && make_map(&mA_lo, a_lo, nA, (int)ks_max, pitch, kBM, bk) &&
          make_map(&mB_hi, b_hi, nB, (int)ks_max, pitch, kBN, bk) && make_map(&mB_lo, b_lo, nB, (int)ks_max, pitch, kBN, bk)))
        return cudaErrorInvalidValue;
    constexpr int smem = Geo<bk>::kSmemBytes;
    e = cudaFuncSetAttribute(kd_umma_kernel<bk>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    int dev = 0, sms = 148;
    if (e == cudaSuccess) e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int grid = n_tiles < sms ? n_tiles : sms;
    for (long long k0 = 0; e == cudaSuccess && k0 < Kdim; k0 += ks_max) {
        const int ks = (int)(Kdim - k0 < ks_max ? Kdim - k0 : ks_max);
        const int kpad = (ks + kMaxBK - 1) / kMaxBK * kMaxBK;
        const dim3 ga((unsigned)((nA + 7) / 8), (unsigned)((kpad + 1023) / 1024)), gb((unsigned)((nB + 7) / 8), ga.y);
        kd_split_kernel<<<ga, 256, 0, s>>>(A, nA, Kdim, k0, ks, kpad, a_hi, a_lo, pitch);
        kd_split_kernel<<<gb, 256, 0, s>>>(B, nB, Kdim, k0, ks, kpad, b_hi, b_lo, pitch);
        UmmaArgs g{d_tiles, n_tiles, kpad / bk, C, nA, nB, ldc, k0 == 0 ? 1 : 0};
        kd_umma_kernel<bk><<<grid, kThreads, smem, s>>>(mA_hi, mA_lo, mB_hi, mB_lo, g);
        e = cudaGetLastError();
    }
    return e;
}

}  // namespace tt
