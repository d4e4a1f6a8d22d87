// tt_gemv.cu - the per-frequency complex matvecs against the precomputed spectrum Fhat
// (steps A2 and B2 of DESIGN.md; "block-diagonal matvec operation in Fourier space" and
// "conjugate-transposed diagonal blocks").  Both kernels stream Fhat from HBM
// exactly once with 128-bit loads that bypass L1; they are bandwidth-bound (1 flop per byte
// in complex64, 0.5 in complex128), so the design goal is bytes in flight, not math.
#include <cstdio>

#include "tt_common.cuh"
#include "tt_internal.h"

namespace tt {

// ---------------------------------------------------------------------------------------
// A2  forward:  partial[w][c][s] = sum_{p in chunk c} Fhat_w[s,p] * xhat_w[p]
//
// One CTA per (frequency w, chunk c of the parameter axis).  The chunk of the input spectrum
// xhat_w is staged once in shared memory and reused for all N_d rows; each warp then owns
// rows s = warp, warp + NWARPS, ...: its 32 lanes sweep the row segment with UNROLL
// independent 128-bit loads in flight per lane, accumulate privately and meet in one
// shuffle reduction per row.  Cross-chunk sums are formed in fixed order by the inverse-FFT
// kernel (no atomics: results are bit-reproducible run to run).
// ---------------------------------------------------------------------------------------
template <typename R, int UNROLL>
__global__ void __launch_bounds__(1024)
gemv_fwd_kernel(const Cx<R>* __restrict__ Fhat, const Cx<R>* __restrict__ xhat, Cx<R>* __restrict__ partial,
                const GemvGeom g) {
    using V = typename Vec16<R>::type;
    constexpr int VN = Vec16<R>::n;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    V* xs = reinterpret_cast<V*>(smem_raw);

    const int w = blockIdx.y, c = blockIdx.x + (int)(g.p_begin / g.chunk);
    const long long p0 = (long long)c * g.chunk;
    const long long rem = g.ldp - p0;
    const int len = rem < g.chunk ? (int)rem : g.chunk;
    const int nvec = len / VN;

    const V* xsrc = reinterpret_cast<const V*>(xhat + (long long)w * g.ldp + p0);
    const int NWARPS = blockDim.x >> 5;
    for (int i = threadIdx.x; i < nvec; i += blockDim.x) xs[i] = xsrc[i];
    __syncthreads();

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int s = warp; s < g.N_d; s += NWARPS) {
        const V* row = reinterpret_cast<const V*>(Fhat + ((long long)w * g.N_d + s) * g.ldp + p0);
        Cx<R> acc0 = mk<R>(R(0), R(0)), acc1 = acc0;
        int i = lane;
        for (; i + (UNROLL - 1) * 32 < nvec; i += UNROLL * 32) {
            V f[UNROLL];
#pragma unroll
            for (int u = 0; u < UNROLL; ++u) f[u] = ldg_stream(row + i + u * 32);
#pragma unroll
            for (int u = 0; u < UNROLL; ++u) {
                const V x = xs[i + u * 32];
#pragma unroll
                for (int e = 0; e < VN; ++e) {
                    if (u & 1) cmac(acc1, Vec16<R>::get(f[u], e), Vec16<R>::get(x, e));
                    else       cmac(acc0, Vec16<R>::get(f[u], e), Vec16<R>::get(x, e));
                }
            }
        }
        for (; i < nvec; i += 32) {
            const V f = ldg_stream(row + i);
            const V x = xs[i];
#pragma unroll
            for (int e = 0; e < VN; ++e) cmac(acc0, Vec16<R>::get(f, e), Vec16<R>::get(x, e));
        }
        const Cx<R> tot = warp_sum(acc0 + acc1);
        if (lane == 0) partial[((long long)w * g.n_chunks + c) * g.N_d + s] = tot;
    }
}

// ---------------------------------------------------------------------------------------
// B2  adjoint:  xout_w[p] = sum_s conj(Fhat_w[s,p]) * dhat_w[s]
//
// One CTA per (frequency w, NT*VN consecutive parameters).  A thread owns one 16-byte column
// vector of p and walks down the N_d rows with UNROLL independent loads in flight; a warp
// reads 512 contiguous bytes of every row.  dhat_w (N_d complex numbers) sits in shared
// memory and is broadcast.  No reduction across threads.
//
// PRODUCER mode (L2R, tt_api.cu run_rmatvec): B3 runs at the same time as a few persistent CTAs that consume the spectrum
// tile by tile (tt_fft.cu fft_c2r_consumer_kernel).  The 1-D grid then runs GROUP by group - l2r_tpg CTA tiles of
// parameters, all frequencies of a group before the next group - so that the spectrum of a group (tens of MB) is complete
// soon after its first store and can wait for its consumer in the L2: Fhat is loaded evict-first, the output stored
// evict-last, and every CTA counts itself into its tile's counter after the store (release by fence + atomic).
// ---------------------------------------------------------------------------------------
template <typename R, int UNROLL, bool L2R = false>
__global__ void __launch_bounds__(512)
gemv_adj_kernel(const Cx<R>* __restrict__ Fhat, const Cx<R>* __restrict__ dhat, Cx<R>* __restrict__ xout,
                const GemvGeom g) {
    using V = typename Vec16<R>::type;
    constexpr int VN = Vec16<R>::n;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    Cx<R>* ds = reinterpret_cast<Cx<R>*>(smem_raw);

    const int NT = blockDim.x;
    const long long rowv = g.ldp / VN;
    int w;
    long long tile;
    if constexpr (L2R) {
        // x -> (group, frequency, tile in group), tile fastest; the last group may hold fewer tiles
        const long long n_tiles = (rowv + NT - 1) / NT;
        const long long per_group = (long long)g.n_f * g.l2r_tpg;
        const long long grp = (long long)blockIdx.x / per_group;
        const long long in_grp = (long long)blockIdx.x - grp * per_group;
        const long long t0 = grp * g.l2r_tpg;
        const int tpg = (int)(n_tiles - t0 < g.l2r_tpg ? n_tiles - t0 : g.l2r_tpg);
        w = (int)(in_grp / tpg);
        tile = t0 + (in_grp - (long long)w * tpg);
    } else {
        w = blockIdx.y;
        tile = blockIdx.x;
    }
    for (int i = threadIdx.x; i < g.N_d; i += NT) ds[i] = dhat[(long long)w * g.N_d + i];
    __syncthreads();

    const long long v = tile * NT + threadIdx.x + (L2R ? 0 : g.p_begin / VN);
    const bool mine = v < (!L2R && g.p_end ? g.p_end / VN : rowv);
    if (!L2R && !mine) return;
    uint64_t pol_in = 0, pol_out = 0;
    if constexpr (L2R) { pol_in = l2_policy_evict_first(); pol_out = l2_policy_evict_last(); }
    auto ld = [&](const V* q) -> V {
        if constexpr (L2R) return ldg_stream(q, pol_in);
        else return ldg_stream(q);
    };
    if (mine) {
        const V* col = reinterpret_cast<const V*>(Fhat + (long long)w * g.N_d * g.ldp) + v;
        Cx<R> acc[VN];
#pragma unroll
        for (int e = 0; e < VN; ++e) acc[e] = mk<R>(R(0), R(0));
        int s = 0;
        for (; s + UNROLL <= g.N_d; s += UNROLL) {
            V f[UNROLL];
#pragma unroll
            for (int u = 0; u < UNROLL; ++u) f[u] = ld(col + (long long)(s + u) * rowv);
#pragma unroll
            for (int u = 0; u < UNROLL; ++u) {
                const Cx<R> dv = ds[s + u];
#pragma unroll
                for (int e = 0; e < VN; ++e) cmac_conj(acc[e], Vec16<R>::get(f[u], e), dv);
            }
        }
        for (; s < g.N_d; ++s) {
            const V f = ld(col + (long long)s * rowv);
            const Cx<R> dv = ds[s];
#pragma unroll
            for (int e = 0; e < VN; ++e) cmac_conj(acc[e], Vec16<R>::get(f, e), dv);
        }
        V* dst = reinterpret_cast<V*>(xout + (long long)w * g.ldp) + v;
        if constexpr (L2R) stg_hint(dst, Vec16<R>::pack(acc[0], acc[VN - 1]), pol_out);
        else *dst = Vec16<R>::pack(acc[0], acc[VN - 1]);
    }
    if constexpr (L2R) {
        __syncthreads();                       // every store of the CTA has been issued ...
        if (threadIdx.x == 0) {
            __threadfence();                   // ... and is visible GPU-wide before the tile's counter moves
            atomicAdd(g.l2r_sync + 2 + tile, 1u);
        }
    }
}

// ---------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------
static int g_fwd_warps = 0, g_adj_threads = 0;
void gemv_debug_set(int fwd_warps, int adj_threads) {
    if (fwd_warps >= 0) g_fwd_warps = fwd_warps;
    if (adj_threads >= 0) g_adj_threads = adj_threads;
}

// Warps per CTA of the forward kernel.  Measured at C3 on B200 (N_d = 100): 10, 16 and 20 warps are within
// 1 % of each other (11.5-11.6 ms), 25 and 32 warps (one CTA per SM) lose 20 %; 16 it is.
static int fwd_warps(int) { return g_fwd_warps ? g_fwd_warps : 16; }

template <typename R>
static cudaError_t fwd_dispatch(const void* Fhat, const void* xhat, void* partial, const GemvGeom& g,
                                cudaStream_t s) {
    constexpr int UN = 8;
    const int NW = g_fwd_warps ? g_fwd_warps : g.warps ? g.warps : fwd_warps(g.N_d);
    auto k = gemv_fwd_kernel<R, UN>;
    const size_t smem = (size_t)g.chunk * sizeof(Cx<R>);
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const long long pe = g.p_end ? g.p_end : g.ldp;
    dim3 grid((unsigned)((pe - g.p_begin + g.chunk - 1) / g.chunk), (unsigned)g.n_f);
    k<<<grid, NW * 32, smem, s>>>(static_cast<const Cx<R>*>(Fhat), static_cast<const Cx<R>*>(xhat),
                                 static_cast<Cx<R>*>(partial), g);
    return cudaGetLastError();
}

template <typename R>
static cudaError_t adj_dispatch(const void* Fhat, const void* dhat, void* xout, const GemvGeom& g,
                                cudaStream_t s) {
    constexpr int UN = 10;
    const int NT = g_adj_threads ? g_adj_threads : 256;
    auto k = g.l2r_sync ? gemv_adj_kernel<R, UN, true> : gemv_adj_kernel<R, UN, false>;
    const size_t smem = (size_t)g.N_d * sizeof(Cx<R>);
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const long long rowv = g.ldp / Vec16<R>::n;
    const long long nv = (g.p_end ? g.p_end : g.ldp) / Vec16<R>::n - g.p_begin / Vec16<R>::n;
    dim3 grid((unsigned)((nv + NT - 1) / NT), (unsigned)g.n_f);
    if (g.l2r_sync) {   // producer mode: the whole parameter axis, group-major 1-D grid
        if (g.p_begin || g.p_end || g.l2r_tpg < 1) return cudaErrorInvalidValue;
        const long long n_cta = ((rowv + NT - 1) / NT) * (long long)g.n_f;
        if (n_cta > 0x7fffffffLL) return cudaErrorInvalidValue;
        grid = dim3((unsigned)n_cta, 1u);
    }
    k<<<grid, NT, smem, s>>>(static_cast<const Cx<R>*>(Fhat), static_cast<const Cx<R>*>(dhat),
                             static_cast<Cx<R>*>(xout), g);
    return cudaGetLastError();
}

int gemv_adj_tile_params(int dt) { return (g_adj_threads ? g_adj_threads : 256) * (dt == 0 ? 2 : 1); }

// What the two launches above look like for geometry g (tt_plan_describe: bench.py ties its ncu figures to this string)
int gemv_describe(int dt, const GemvGeom& g, char* buf, size_t n) {
    const int NW = g_fwd_warps ? g_fwd_warps : g.warps ? g.warps : fwd_warps(g.N_d);
    const int NT = g_adj_threads ? g_adj_threads : 256;
    const int vn = dt == 0 ? 2 : 1;
    const long long pe = g.p_end ? g.p_end : g.ldp;
    return snprintf(buf, n,
                    "A2 gemv_fwd_kernel<%s,8> grid=(%lld,%d) block=%d smem=%zu chunk=%d | "
                    "B2 gemv_adj_kernel<%s,10> grid=(%lld,%d) block=%d smem=%zu",
                    dt == 0 ? "float" : "double", (pe - g.p_begin + g.chunk - 1) / g.chunk, g.n_f, NW * 32,
                    (size_t)g.chunk * (dt == 0 ? 8 : 16), g.chunk, dt == 0 ? "float" : "double",
                    ((pe - g.p_begin) / vn + NT - 1) / NT, g.n_f, NT, (size_t)g.N_d * (dt == 0 ? 8 : 16));
}

cudaError_t gemv_fwd_launch(int dt, const void* Fhat, const void* xhat, void* partial, const GemvGeom& g,
                            cudaStream_t s) {
    return dt == 0 ? fwd_dispatch<float>(Fhat, xhat, partial, g, s) : fwd_dispatch<double>(Fhat, xhat, partial, g, s);
}
cudaError_t gemv_adj_launch(int dt, const void* Fhat, const void* dhat, void* xout, const GemvGeom& g,
                            cudaStream_t s) {
    return dt == 0 ? adj_dispatch<float>(Fhat, dhat, xout, g, s) : adj_dispatch<double>(Fhat, dhat, xout, g, s);
}

}  // namespace tt
