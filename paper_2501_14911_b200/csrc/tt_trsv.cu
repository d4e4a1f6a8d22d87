// tt_trsv.cu - the two triangular solves of the online phase, K^{-1} b = L^{-T} (L^{-1} b) with the
// Cholesky factor K = L L^T of the data-space matrix K = Gamma_noise + F G* ("This matrix can be
// Cholesky-factorized offline, and triangular solves are done in the online phase", PAPER.md:294;
// 20 ms of the 53 ms online inference on the paper's system).
//
// A dense triangular solve is one pass over the factor (n^2/2 doubles: 2.4 GB at the paper's
// n = N_d N_t = 24 500) plus a dependency chain of n/NB block steps.  The design goal is to make the
// chain step as short as one L2 round trip plus a handful of instructions, and to let everything that
// is not on the chain stream at HBM speed behind it:
//
//   * At plan time the factor is rescaled by its diagonal blocks, Lt = D^{-1} L with
//     D = blockdiag(L_II), NB = 64: Lt has identity diagonal blocks, so that
//          L^{-1} b   = Lt^{-1} (D^{-1} b)            L^{-T} y = D^{-T} (Lt^{-T} y)
//     and the chain of either solve is a pure block recurrence with NO diagonal solve on it:
//          forward   y_I  = bt_I - sum_{J<I} Lt_IJ   y_J          (bt = D^{-1} b, fully parallel pre-step)
//          backward  xt_I = y_I  - sum_{J>I} Lt_JI^T xt_J         (x  = D^{-T} xt, fully parallel post-step)
//     Only the strictly lower blocks of Lt are stored (half the memory of the square factor), each
//     64 x 64 block contiguous (32 KB) and the blocks of one block row one after the other, so that
//     every CTA of the forward solve reads ONE sequential stream; plus the NB x NB inverses D_I^{-1}.
//   * One CTA per block row (forward) / block column (backward).  A CTA takes its block index from an
//     atomic ticket, so a CTA only ever waits for blocks owned by CTAs that have already started:
//     no co-residency assumption, no deadlock.
//   * Data is its own flag: the solution vector is pre-filled with a NaN bit pattern that no
//     arithmetic produces; a producer publishes 64-bit values with plain stores and consumers spin on
//     the very values they need (relaxed loads that bypass L1).  Every 8-byte value is self-validating,
//     so the chain needs no fence and no separate flag round trip.
//   * Each warp owns 8 rows (forward) or 8 block rows of the reduction (backward), keeps U = 2 blocks
//     (8 KB per warp, 64 KB per CTA) of Lt in flight in registers and never synchronises with the rest
//     of the CTA inside the streaming loop.
// All sums have a fixed order: results are bit-reproducible run to run.
#include "tt_common.cuh"
#include "tt_internal.h"

namespace tt {

namespace {

constexpr int NB = kTrsvNB;     // block order
constexpr int RW = 8;           // rows per warp
constexpr int NTHREADS = (NB / RW) * 32;
constexpr unsigned long long kSentinel = 0x7FF4A5A5DEADBEEFULL;  // signalling-NaN payload: "not yet computed"

__device__ __forceinline__ bool is_sentinel(double v) { return (unsigned long long)__double_as_longlong(v) == kSentinel; }

// value to publish: a computed number can never carry the sentinel payload (arithmetic NaNs are canonical),
// but an input may; map it to the canonical NaN so that a consumer cannot hang on it.
__device__ __forceinline__ double publishable(double v) {
    return is_sentinel(v) ? __longlong_as_double(0x7FF8000000000000LL) : v;
}

__device__ __forceinline__ double2 ld_poll2(const double* p) {
    double2 v;
    asm volatile("ld.relaxed.gpu.global.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_publish(double* p, double v) {
    asm volatile("st.relaxed.gpu.global.f64 [%0], %1;" ::"l"(p), "d"(v) : "memory");
}

// Sum of acc[r] over the 32 lanes for r = 0..7 with 9 exchanges: afterwards the lanes with (lane & 3) == 0
// hold the total of row  r = 4*bit4(lane) + 2*bit3(lane) + bit2(lane).
__device__ __forceinline__ double reduce8(const double (&acc)[RW], int lane) {
    double a4[4], a2[2];
    {
        const bool hi = lane & 16;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const double send = hi ? acc[i] : acc[i + 4];
            const double keep = hi ? acc[i + 4] : acc[i];
            a4[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
        }
    }
    {
        const bool hi = lane & 8;
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            const double send = hi ? a4[i] : a4[i + 2];
            const double keep = hi ? a4[i + 2] : a4[i];
            a2[i] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
        }
    }
    double a1;
    {
        const bool hi = lane & 4;
        const double send = hi ? a2[0] : a2[1];
        const double keep = hi ? a2[1] : a2[0];
        a1 = keep + __shfl_xor_sync(0xffffffffu, send, 4);
    }
    a1 += __shfl_xor_sync(0xffffffffu, a1, 2);
    a1 += __shfl_xor_sync(0xffffffffu, a1, 1);
    return a1;
}

// ---------------------------------------------------------------------------------------
// forward chain:  y_I = bt_I - sum_{J<I} Lt_IJ y_J
// ---------------------------------------------------------------------------------------
// Block (I, J), J < I, of Lt: NB x NB doubles, row-major, contiguous (32 KB); the blocks of block row I follow
// each other, so that the forward solve reads one sequential stream per CTA.
__device__ __forceinline__ size_t blk_off(int I, int J) {
    return (size_t)NB * NB * ((size_t)I * (size_t)(I - 1) / 2 + (size_t)J);
}

// ---------------------------------------------------------------------------------------
// forward chain:  y_I = bt_I - sum_{J<I} Lt_IJ y_J
// Warp w owns rows 8w..8w+7 (4 KB contiguous per block); lane owns columns 2*lane, 2*lane+1.
// ---------------------------------------------------------------------------------------
template <int U>
__global__ void __launch_bounds__(NTHREADS, 2)
trsv_fwd_kernel(const double* __restrict__ Lt, const double* __restrict__ bt, double* y, unsigned* ticket) {
    __shared__ int sI;
    if (threadIdx.x == 0) sI = (int)atomicAdd(ticket, 1u);
    __syncthreads();
    const int I = sI;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const double* rowp = Lt + blk_off(I, 0) + (size_t)(warp * RW) * NB + 2 * lane;
    // the right-hand side of the row this lane will publish, fetched before the chain needs it
    const int my_r = ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1);
    const size_t my_row = (size_t)I * NB + warp * RW + my_r;
    const double my_bt = bt[my_row];

    double acc[RW];
#pragma unroll
    for (int r = 0; r < RW; ++r) acc[r] = 0.0;
    double2 buf[U][RW];
#pragma unroll
    for (int u = 0; u < U; ++u)
        if (u < I) {
#pragma unroll
            for (int r = 0; r < RW; ++r)
                buf[u][r] = ldg_stream(reinterpret_cast<const double2*>(rowp + (size_t)u * NB * NB + r * NB));
        }
    for (int J0 = 0; J0 < I; J0 += U) {
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int J = J0 + u;
            if (J < I) {
                const double* yp = y + (size_t)J * NB + 2 * lane;
                // Every waiting warp spins at full rate: a back-off (__nanosleep) for the CTAs far from the chain
                // head and a look-ahead poll of y_{J+1} were both measured slower (B200, n = 4096 / 24 500).
                double2 yv;
#pragma unroll 1
                do { yv = ld_poll2(yp); } while (is_sentinel(yv.x) || is_sentinel(yv.y));   // one load per attempt
#pragma unroll
                for (int r = 0; r < RW; ++r) {
                    acc[r] = fma(buf[u][r].x, yv.x, acc[r]);
                    acc[r] = fma(buf[u][r].y, yv.y, acc[r]);
                }
                if (J + U < I) {
#pragma unroll
                    for (int r = 0; r < RW; ++r)
                        buf[u][r] = ldg_stream(reinterpret_cast<const double2*>(rowp + (size_t)(J + U) * NB * NB + r * NB));
                }
            }
        }
    }
    const double tot = reduce8(acc, lane);
    // Publish the 64 values of the block row with ONE warp-wide store: when the eight warps publish their eight rows
    // each, a consumer's poll usually lands in the middle and pays a second L2 round trip (~0.3 us) for the rest.
    __shared__ __align__(16) double ys[NB];
    if ((lane & 3) == 0) ys[warp * RW + my_r] = publishable(my_bt - tot);
    __syncthreads();
    if (warp == 0) {
        const double2 v = *reinterpret_cast<const double2*>(ys + 2 * lane);
        asm volatile("st.relaxed.gpu.global.v2.f64 [%0], {%1, %2};" ::"l"(y + (size_t)I * NB + 2 * lane), "d"(v.x), "d"(v.y) : "memory");
    }
}

// ---------------------------------------------------------------------------------------
// backward chain:  xt_I = y_I - sum_{J>I} Lt_JI^T xt_J
// Warp w sums rows 8w..8w+7 of every block (J, I); lane owns columns 2*lane, 2*lane+1.
// ---------------------------------------------------------------------------------------
template <int U>
__global__ void __launch_bounds__(NTHREADS, 2)
trsv_bwd_kernel(const double* __restrict__ Lt, const double* __restrict__ yin, double* xt, unsigned* ticket, int nblk) {
    __shared__ int sI;
    __shared__ double part[NB / RW][NB];
    if (threadIdx.x == 0) sI = nblk - 1 - (int)atomicAdd(ticket, 1u);
    __syncthreads();
    const int I = sI;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nJ = nblk - 1 - I;  // blocks below the diagonal in block column I; the t-th visited is J = nblk-1-t
    const double my_y = threadIdx.x < NB ? yin[(size_t)I * NB + threadIdx.x] : 0.0;

    auto blk = [&](int t) { return Lt + blk_off(nblk - 1 - t, I) + (size_t)(warp * RW) * NB + 2 * lane; };
    double2 acc = make_double2(0.0, 0.0);
    double2 buf[U][RW];
#pragma unroll
    for (int u = 0; u < U; ++u)
        if (u < nJ) {
            const double* p = blk(u);
#pragma unroll
            for (int r = 0; r < RW; ++r) buf[u][r] = ldg_stream(reinterpret_cast<const double2*>(p + r * NB));
        }
    for (int t0 = 0; t0 < nJ; t0 += U) {
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int t = t0 + u;
            if (t < nJ) {
                const int J = nblk - 1 - t;
                const double* xp = xt + (size_t)J * NB + warp * RW;
                double2 xv[RW / 2];
                bool ok;
#pragma unroll 1
                do {   // the four loads of one attempt are in flight together
#pragma unroll
                    for (int r = 0; r < RW / 2; ++r) xv[r] = ld_poll2(xp + 2 * r);
                    ok = true;
#pragma unroll
                    for (int r = 0; r < RW / 2; ++r) ok = ok && !is_sentinel(xv[r].x) && !is_sentinel(xv[r].y);
                } while (!ok);
#pragma unroll
                for (int r = 0; r < RW / 2; ++r) {
                    acc.x = fma(buf[u][2 * r].x, xv[r].x, acc.x);
                    acc.y = fma(buf[u][2 * r].y, xv[r].x, acc.y);
                    acc.x = fma(buf[u][2 * r + 1].x, xv[r].y, acc.x);
                    acc.y = fma(buf[u][2 * r + 1].y, xv[r].y, acc.y);
                }
                if (t + U < nJ) {
                    const double* p = blk(t + U);
#pragma unroll
                    for (int r = 0; r < RW; ++r) buf[u][r] = ldg_stream(reinterpret_cast<const double2*>(p + r * NB));
                }
            }
        }
    }
    part[warp][2 * lane] = acc.x;
    part[warp][2 * lane + 1] = acc.y;
    __syncthreads();
    // (two warps publish 256 bytes each; a single warp-wide store as in the forward kernel was measured slower here)
    if (threadIdx.x < NB) {
        double s = 0.0;
#pragma unroll
        for (int w = 0; w < NB / RW; ++w) s += part[w][threadIdx.x];
        st_publish(xt + (size_t)I * NB + threadIdx.x, publishable(my_y - s));
    }
}

// ---------------------------------------------------------------------------------------
// pre-step:  bt = D^{-1} b (b == nullptr: skipped), reset of the two self-flagging vectors and tickets
// post-step: x = D^{-T} xt
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
trsv_pre_kernel(const double* __restrict__ Dinv, const double* __restrict__ b, double* __restrict__ bt,
                double* y, double* xt, unsigned* ticket, long long n) {
    const int I = blockIdx.x, tid = threadIdx.x;
    __shared__ double bs[NB];
    const double sent = __longlong_as_double((long long)kSentinel);
    if (tid < NB) {
        const long long row = (long long)I * NB + tid;
        y[row] = sent;
        xt[row] = sent;
        if (b) bs[tid] = row < n ? b[row] : 0.0;
    }
    if (I == 0 && tid == 0) { ticket[0] = 0u; ticket[1] = 0u; }
    if (!b) return;
    __syncthreads();
    const int r = tid >> 2, q = tid & 3;
    const double* drow = Dinv + ((size_t)I * NB + r) * NB + q * 16;
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < 16; ++c) s = fma(drow[c], bs[q * 16 + c], s);
    s += __shfl_xor_sync(0xffffffffu, s, 1);
    s += __shfl_xor_sync(0xffffffffu, s, 2);
    if (q == 0) bt[(size_t)I * NB + r] = s;
}

__global__ void __launch_bounds__(256)
trsv_post_kernel(const double* __restrict__ Dinv, const double* __restrict__ xt, double* __restrict__ x, long long n) {
    const int I = blockIdx.x, tid = threadIdx.x;
    __shared__ double xs[NB];
    __shared__ double part[4][NB];
    if (tid < NB) xs[tid] = xt[(size_t)I * NB + tid];
    __syncthreads();
    const int c = tid & (NB - 1), q = tid / NB;  // q = 0..3: rows q*16 .. q*16+15
    const double* d = Dinv + ((size_t)I * NB + q * 16) * NB + c;
    double s = 0.0;
#pragma unroll
    for (int r = 0; r < 16; ++r) s = fma(d[(size_t)r * NB], xs[q * 16 + r], s);
    part[q][c] = s;
    __syncthreads();
    if (tid < NB) {
        const long long row = (long long)I * NB + tid;
        if (row < n) x[row] = (part[0][tid] + part[1][tid]) + (part[2][tid] + part[3][tid]);
    }
}

__global__ void trsv_copy_kernel(const double* __restrict__ src, double* __restrict__ dst, long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[i] = src[i];
}

// ---------------------------------------------------------------------------------------
// plan time: D_I^{-1} and Lt = D^{-1} L (packed strictly-lower blocks)
// src: rows [row0, row0 + nrows) of the row-major factor, pitch ld; row0 is a multiple of NB.
// ---------------------------------------------------------------------------------------
// One CTA of 64 threads per diagonal block: thread c solves L_II X[:,c] = e_c by forward substitution.
__global__ void __launch_bounds__(NB)
trsv_dinv_kernel(const double* __restrict__ src, long long ld, long long row0, long long n, double* __restrict__ Dinv,
                 int* __restrict__ bad) {
    __shared__ double Ls[NB][NB + 1];
    const int Il = blockIdx.x;                      // block row within the slab
    const long long g0 = row0 + (long long)Il * NB;  // first global row/col of the diagonal block
    const int c = threadIdx.x;
    for (int r = 0; r < NB; ++r) {
        const long long gr = g0 + r, gc = g0 + c;
        double v = (r == c) ? 1.0 : 0.0;            // padding beyond n: identity
        if (gr < n && gc < n) v = (c <= r) ? src[(size_t)(gr - row0) * ld + gc] : 0.0;
        Ls[r][c] = v;
    }
    __syncthreads();
    {
        const double dg = Ls[c][c];
        if (!(dg > 0.0) || !(dg < 1.0e300)) atomicExch(bad, 1);   // Cholesky factors have a positive finite diagonal
    }
    double xc[NB];                                   // column c of the inverse (one-time kernel: local memory is fine)
    for (int r = 0; r < NB; ++r) {
        double s = (r == c) ? 1.0 : 0.0;
        for (int q = c; q < r; ++q) s = fma(-Ls[r][q], xc[q], s);   // X is lower triangular: X[q][c] = 0 for q < c
        xc[r] = (r >= c) ? s / Ls[r][r] : 0.0;
    }
    double* out = Dinv + (size_t)(g0 / NB) * NB * NB;
    for (int r = 0; r < NB; ++r) out[(size_t)r * NB + c] = xc[r];
}

// Lt_IJ = D_I^{-1} L_IJ, one CTA of 256 threads per block (J = blockIdx.x < I = I0 + blockIdx.y).
__global__ void __launch_bounds__(256)
trsv_scale_kernel(const double* __restrict__ src, long long ld, long long row0, long long n,
                  const double* __restrict__ Dinv, double* __restrict__ Lt) {
    const int I = (int)(row0 / NB) + blockIdx.y, J = blockIdx.x;
    if (J >= I) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double (*Ds)[NB + 1] = reinterpret_cast<double (*)[NB + 1]>(smem_raw);
    double (*Ls)[NB] = reinterpret_cast<double (*)[NB]>(smem_raw + sizeof(double) * NB * (NB + 1));
    const int tid = threadIdx.x;
    const double* Di = Dinv + (size_t)I * NB * NB;
    for (int e = tid; e < NB * NB; e += 256) {
        const int r = e / NB, c = e % NB;
        Ds[r][c] = Di[e];
        const long long gr = (long long)I * NB + r, gc = (long long)J * NB + c;
        Ls[r][c] = (gr < n) ? src[(size_t)(gr - row0) * ld + gc] : 0.0;
    }
    __syncthreads();
    // thread -> 4 rows x 4 columns
    const int r0 = (tid / 16) * 4, c0 = (tid % 16) * 4;
    double o[4][4] = {};
    for (int q = 0; q < NB; ++q) {
        double a[4], b[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) { a[i] = Ds[r0 + i][q]; b[i] = Ls[q][c0 + i]; }
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) o[i][j] = fma(a[i], b[j], o[i][j]);
    }
    double* dst = Lt + blk_off(I, J);
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) dst[(size_t)(r0 + i) * NB + c0 + j] = o[i][j];
}

}  // namespace

cudaError_t trsv_prepare_launch(const double* src, long long ld, long long row0, long long nrows, long long n,
                                double* Dinv, double* Lt, int* bad, cudaStream_t s) {
    const int nb_rows = (int)((nrows + NB - 1) / NB);
    if (nb_rows < 1) return cudaSuccess;
    trsv_dinv_kernel<<<nb_rows, NB, 0, s>>>(src, ld, row0, n, Dinv, bad);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const int Imax = (int)(row0 / NB) + nb_rows - 1;  // largest block row of the slab
    if (Imax >= 1) {
        constexpr int smem = (int)(sizeof(double) * (NB * (NB + 1) + NB * NB));
        e = cudaFuncSetAttribute(trsv_scale_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
        // gridDim.x = number of column blocks of the longest row; CTAs with J >= I exit at once
        for (int y0 = 0; y0 < nb_rows; y0 += 32768) {
            const int ny = nb_rows - y0 < 32768 ? nb_rows - y0 : 32768;
            dim3 grid((unsigned)Imax, (unsigned)ny);
            trsv_scale_kernel<<<grid, 256, smem, s>>>(src + (size_t)y0 * NB * ld, ld, row0 + (long long)y0 * NB, n, Dinv, Lt);
            e = cudaGetLastError();
            if (e != cudaSuccess) return e;
        }
    }
    return cudaSuccess;
}

cudaError_t trsv_pre_launch(const TrsvGeom& g, const double* b, cudaStream_t s) {
    trsv_pre_kernel<<<g.nblk, 256, 0, s>>>(g.Dinv, b, g.bt, g.y, g.xt, g.ticket, g.n);
    return cudaGetLastError();
}
static int g_trsv_U = 0;
void trsv_debug_set_U(int U) { g_trsv_U = U; }

cudaError_t trsv_fwd_launch(const TrsvGeom& g, cudaStream_t s) {
    if (g_trsv_U == 3) trsv_fwd_kernel<3><<<g.nblk, NTHREADS, 0, s>>>(g.Lt, g.bt, g.y, g.ticket);
    else if (g_trsv_U == 1) trsv_fwd_kernel<1><<<g.nblk, NTHREADS, 0, s>>>(g.Lt, g.bt, g.y, g.ticket);
    else trsv_fwd_kernel<2><<<g.nblk, NTHREADS, 0, s>>>(g.Lt, g.bt, g.y, g.ticket);
    return cudaGetLastError();
}
cudaError_t trsv_bwd_launch(const TrsvGeom& g, const double* yin, cudaStream_t s) {
    if (g_trsv_U == 1) trsv_bwd_kernel<1><<<g.nblk, NTHREADS, 0, s>>>(g.Lt, yin, g.xt, g.ticket + 1, g.nblk);
    else if (g_trsv_U == 2) trsv_bwd_kernel<2><<<g.nblk, NTHREADS, 0, s>>>(g.Lt, yin, g.xt, g.ticket + 1, g.nblk);
    else trsv_bwd_kernel<3><<<g.nblk, NTHREADS, 0, s>>>(g.Lt, yin, g.xt, g.ticket + 1, g.nblk);   // default: three blocks in flight
    return cudaGetLastError();
}
cudaError_t trsv_post_launch(const TrsvGeom& g, double* x, cudaStream_t s) {
    trsv_post_kernel<<<g.nblk, 256, 0, s>>>(g.Dinv, g.xt, x, g.n);
    return cudaGetLastError();
}
cudaError_t trsv_copy_launch(const double* src, double* dst, long long n, cudaStream_t s) {
    trsv_copy_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(src, dst, n);
    return cudaGetLastError();
}

}  // namespace tt
