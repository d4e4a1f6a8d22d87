// tt_gemm.cu - k right-hand sides at once: the per-frequency products become complex GEMMs
//     forward   Dhat_w [N_d x k] = Fhat_w   [N_d x N_m] * Xhat_w [N_m x k]
//     adjoint   Xhat_w [N_m x k] = Fhat_w^H [N_m x N_d] * Dhat_w [N_d x k]
// (step D of DESIGN.md; the many-matvec workloads of PAPER.md:296, 407, 421-423).  This is the one
// place on the path that is a dense contraction (16 flop per Fhat byte at k = 32), so it runs on
// the FP64 tensor pipe: mma.sync m8n8k4 f64 (SASS DMMA.8x8x4) - tcgen05 has no FP64 kind.  A
// complex product is four real DMMAs on the (re, im) halves of the interleaved operands:
//     Cr += Ar*Br;  Cr += (-Ai)*Bi;  Ci += Ar*Bi;  Ci += Ai*Br.
// One 16-byte complex element per thread IS the DMMA fragment pair (re-fragment, im-fragment):
//     A (8x4, row):  row = lane/4, col = lane%4      B (4x8, col):  row = lane%4, col = lane/4
//     C (8x8):       row = lane/4, cols = 2*(lane%4) + {0,1}
#include "tt_common.cuh"
#include "tt_internal.h"

namespace tt {

__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
constexpr int kFwdKP = 32;            // parameters per pipeline stage (8 DMMA k-steps)
constexpr int kFwdApitch = kFwdKP + 4;  // complex elements; +4 keeps the 8-lane LDS.128 phases conflict-free
constexpr int kFwdRows = 64;          // sensors per CTA (4 warps x 2 m-tiles x 8)

// ---------------------------------------------------------------------------------------
// forward: partial[((w*nsplit + c)*N_d + s)*k + r] = sum_{p in split c} Fhat_w[s,p] Xhat_w[p,r]
// grid (nsplit, n_f, ceil(N_d/64)), 128 threads; each warp 16 sensors x 8*NN columns.
// Both operands go through a 2-stage cp.async shared-memory pipeline.
// ---------------------------------------------------------------------------------------
template <int NN>
__global__ void __launch_bounds__(128, 2)
gemm_fwd_kernel(const c128* __restrict__ Fhat, const c128* __restrict__ Xhat, c128* __restrict__ partial,
                const GemmGeom g, const int r0, const int kk) {
    constexpr int BP = 8 * NN + 2;  // B pitch in complex elements
    extern __shared__ __align__(16) unsigned char smem_raw[];
    c128* As = reinterpret_cast<c128*>(smem_raw);                    // [2][64][kFwdApitch]
    c128* Bs = As + 2 * kFwdRows * kFwdApitch;                       // [2][kFwdKP][BP]

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int w = blockIdx.y, c = blockIdx.x, s0 = blockIdx.z * kFwdRows;
    const long long p_lo = (long long)c * g.p_per_split;
    long long p_hi = p_lo + g.p_per_split;
    if (p_hi > g.N_m) p_hi = g.N_m;
    const int n_it = p_hi > p_lo ? (int)((p_hi - p_lo + kFwdKP - 1) / kFwdKP) : 0;

    const c128* Abase = Fhat + ((long long)w * g.N_d + s0) * g.ldp;
    const c128* Bbase = Xhat + (long long)w * g.ldx + r0;

    auto load_stage = [&](int st, int it) {
        const long long p0 = p_lo + (long long)it * kFwdKP;
        c128* a = As + st * kFwdRows * kFwdApitch;
        // A tile: 64 sensors x 32 parameters, 512 contiguous bytes per sensor row
#pragma unroll
        for (int i = 0; i < (kFwdRows * kFwdKP) / 128; ++i) {
            const int e = i * 128 + tid, row = e / kFwdKP, col = e % kFwdKP;
            const bool ok = (s0 + row < g.N_d) && (p0 + col < p_hi);
            cp_async16(a + row * kFwdApitch + col, ok ? Abase + (long long)row * g.ldp + p0 + col : Abase, ok);
        }
        // B tile: 32 parameters x kk columns
        c128* b = Bs + st * kFwdKP * BP;
#pragma unroll
        for (int i = 0; i < (kFwdKP * 8 * NN) / 128; ++i) {
            const int e = i * 128 + tid, row = e / (8 * NN), col = e % (8 * NN);
            const bool ok = (p0 + row < p_hi) && (col < kk);
            cp_async16(b + row * BP + col, ok ? Bbase + (p0 + row) * (long long)g.k + col : Bbase, ok);
        }
    };

    double cr[2][NN][2], ci[2][NN][2];
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
        for (int nt = 0; nt < NN; ++nt) { cr[mt][nt][0] = cr[mt][nt][1] = ci[mt][nt][0] = ci[mt][nt][1] = 0.0; }

    if (n_it > 0) load_stage(0, 0);
    cp_async_commit();
    for (int it = 0; it < n_it; ++it) {
        cp_async_wait<0>();
        __syncthreads();
        if (it + 1 < n_it) load_stage((it + 1) & 1, it + 1);
        cp_async_commit();
        const c128* a = As + (it & 1) * kFwdRows * kFwdApitch + (warp * 16 + (lane >> 2)) * kFwdApitch + (lane & 3);
        const c128* b = Bs + (it & 1) * kFwdKP * BP + (lane & 3) * BP + (lane >> 2);
#pragma unroll
        for (int t = 0; t < kFwdKP / 4; ++t) {
            c128 af[2], bf[NN];
#pragma unroll
            for (int mt = 0; mt < 2; ++mt) af[mt] = a[mt * 8 * kFwdApitch + 4 * t];
#pragma unroll
            for (int nt = 0; nt < NN; ++nt) bf[nt] = b[4 * t * BP + nt * 8];
#pragma unroll
            for (int mt = 0; mt < 2; ++mt)
#pragma unroll
                for (int nt = 0; nt < NN; ++nt) {
                    dmma(cr[mt][nt][0], cr[mt][nt][1], af[mt].re, bf[nt].re);
                    dmma(cr[mt][nt][0], cr[mt][nt][1], -af[mt].im, bf[nt].im);
                    dmma(ci[mt][nt][0], ci[mt][nt][1], af[mt].re, bf[nt].im);
                    dmma(ci[mt][nt][0], ci[mt][nt][1], af[mt].im, bf[nt].re);
                }
        }
    }

    // epilogue: two consecutive complex outputs per thread and tile
#pragma unroll
    for (int mt = 0; mt < 2; ++mt) {
        const int s = s0 + warp * 16 + mt * 8 + (lane >> 2);
        if (s >= g.N_d) continue;
        c128* dst = partial + (((long long)w * g.split + c) * g.N_d + s) * g.k + r0;
#pragma unroll
        for (int nt = 0; nt < NN; ++nt) {
            const int r = nt * 8 + (lane & 3) * 2;
            if (r < kk) dst[r] = mk<double>(cr[mt][nt][0], ci[mt][nt][0]);
            if (r + 1 < kk) dst[r + 1] = mk<double>(cr[mt][nt][1], ci[mt][nt][1]);
        }
    }
}

// ---------------------------------------------------------------------------------------
// adjoint: Xout_w[p, r] = sum_s conj(Fhat_w[s,p]) Dhat_w[s, r]
// grid (ceil(N_m/256), n_f), 256 threads; a warp owns 8 parameters x 8*NN columns at a time and
// walks down the sensors; its A fragments come straight from global memory (4 sensor rows x
// 128 contiguous bytes per load instruction, read once), Dhat_w is staged in shared memory.
//     Cr += Fr*Dr;  Cr += Fi*Di;  Ci += Fr*Di;  Ci += (-Fi)*Dr
// ---------------------------------------------------------------------------------------
constexpr int kAdjSB = 64;    // sensors per shared-memory block of Dhat
constexpr int kAdjPT = 256;   // parameters per CTA (4 rounds of 8 warps x 8)

// MT = m-tiles (8 parameters each) per warp.  MT = 2 (four warps, like the forward kernel: a B fragment read from shared
// memory feeds two DMMA groups) or MT = 1 (eight warps).  Either way a round covers 64 parameters of the CTA's 256.
template <int NN, int MT>
__global__ void __launch_bounds__(256 / MT, MT == 2 ? 3 : 2)
gemm_adj_kernel(const c128* __restrict__ Fhat, const c128* __restrict__ Dhat, c128* __restrict__ Xout,
                const GemmGeom g, const int r0, const int kk) {
    constexpr int BP = 8 * NN + 2, NTH = 256 / MT;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    c128* Ds = reinterpret_cast<c128*>(smem_raw);  // [kAdjSB][BP]

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int w = blockIdx.y;
    const long long pblk = (long long)blockIdx.x * kAdjPT;
    const c128* Fw = Fhat + (long long)w * g.N_d * g.ldp;
    const c128* Dw = Dhat + (long long)w * g.N_d * g.k + r0;

    auto stage_d = [&](int sb) {
        for (int e = tid; e < kAdjSB * 8 * NN; e += NTH) {
            const int row = e / (8 * NN), col = e % (8 * NN);
            c128 v = mk<double>(0.0, 0.0);
            if (sb + row < g.N_d && col < kk) v = Dw[(long long)(sb + row) * g.k + col];
            Ds[row * BP + col] = v;
        }
    };
    const bool single = g.N_d <= kAdjSB;  // Dhat_w fits one shared-memory block: stage it once
    if (single) { stage_d(0); __syncthreads(); }

    for (int rd = 0; rd < kAdjPT / 64; ++rd) {  // rounds of 64 parameters: (8 / MT) warps x MT m-tiles x 8
        long long p[MT];
        bool pok[MT];
#pragma unroll
        for (int mt = 0; mt < MT; ++mt) {
            p[mt] = pblk + rd * 64 + (warp * MT + mt) * 8 + (lane >> 2);
            pok[mt] = p[mt] < g.N_m;
        }
        double cr[MT][NN][2], ci[MT][NN][2];
#pragma unroll
        for (int mt = 0; mt < MT; ++mt)
#pragma unroll
            for (int nt = 0; nt < NN; ++nt) { cr[mt][nt][0] = cr[mt][nt][1] = ci[mt][nt][0] = ci[mt][nt][1] = 0.0; }

        for (int sb = 0; sb < g.N_d; sb += kAdjSB) {
            if (!single) { __syncthreads(); stage_d(sb); __syncthreads(); }
            const int ns = g.N_d - sb < kAdjSB ? g.N_d - sb : kAdjSB;
            const int nsteps = (ns + 3) / 4;
            const c128* row = Fw + (long long)(sb + (lane & 3)) * g.ldp;
            // software pipeline over batches of BK k-steps: the A fragments of batch b+1 are in flight
            // while the DMMAs of batch b issue
            constexpr int BK = MT == 1 ? 4 : 2;
            auto load_batch = [&](c128 (&af)[MT][BK], int t0) {
#pragma unroll
                for (int u = 0; u < BK; ++u) {
                    const int t = t0 + u;
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt) {
                        af[mt][u] = mk<double>(0.0, 0.0);
                        if (pok[mt] && t < nsteps && sb + 4 * t + (lane & 3) < g.N_d) {
                            const double2 v = ldg_stream(reinterpret_cast<const double2*>(row + (long long)(4 * t) * g.ldp + p[mt]));
                            af[mt][u] = mk<double>(v.x, v.y);
                        }
                    }
                }
            };
            auto mma_batch = [&](const c128 (&af)[MT][BK], int t0) {
#pragma unroll
                for (int u = 0; u < BK; ++u) {
                    const int t = t0 + u;
                    if (t < nsteps) {
                        const c128* b = Ds + (4 * t + (lane & 3)) * BP + (lane >> 2);
#pragma unroll
                        for (int nt = 0; nt < NN; ++nt) {
                            const c128 bf = b[nt * 8];
#pragma unroll
                            for (int mt = 0; mt < MT; ++mt) {
                                dmma(cr[mt][nt][0], cr[mt][nt][1], af[mt][u].re, bf.re);
                                dmma(cr[mt][nt][0], cr[mt][nt][1], af[mt][u].im, bf.im);
                                dmma(ci[mt][nt][0], ci[mt][nt][1], af[mt][u].re, bf.im);
                                dmma(ci[mt][nt][0], ci[mt][nt][1], -af[mt][u].im, bf.re);
                            }
                        }
                    }
                }
            };
            c128 a0[MT][BK], a1[MT][BK];
            load_batch(a0, 0);
            for (int t0 = 0; t0 < nsteps; t0 += 2 * BK) {
                load_batch(a1, t0 + BK);
                mma_batch(a0, t0);
                load_batch(a0, t0 + 2 * BK);
                mma_batch(a1, t0 + BK);
            }
        }
#pragma unroll
        for (int mt = 0; mt < MT; ++mt) {
            if (!pok[mt]) continue;
            c128* dst = Xout + (long long)w * g.ldx + p[mt] * g.k + r0;
#pragma unroll
            for (int nt = 0; nt < NN; ++nt) {
                const int r = nt * 8 + (lane & 3) * 2;
                if (r < kk) dst[r] = mk<double>(cr[mt][nt][0], ci[mt][nt][0]);
                if (r + 1 < kk) dst[r + 1] = mk<double>(cr[mt][nt][1], ci[mt][nt][1]);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------
template <int NN>
static cudaError_t fwd_launch_nn(const c128* F, const c128* X, c128* P, const GemmGeom& g, int r0, int kk,
                                 cudaStream_t s) {
    auto k = gemm_fwd_kernel<NN>;
    const size_t smem = (size_t)(2 * kFwdRows * kFwdApitch + 2 * kFwdKP * (8 * NN + 2)) * sizeof(c128);
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    dim3 grid((unsigned)g.split, (unsigned)g.n_f, (unsigned)((g.N_d + kFwdRows - 1) / kFwdRows));
    k<<<grid, 128, smem, s>>>(F, X, P, g, r0, kk);
    return cudaGetLastError();
}

static int g_adj_mt = 2;   // m-tiles per warp of the adjoint kernel (debug key "gemm_adj_mt"; 2 measured 2.3% faster on C4)
void gemm_debug_set_adj(int mt) { g_adj_mt = mt == 1 ? 1 : 2; }

template <int NN>
static cudaError_t adj_launch_nn(const c128* F, const c128* D, c128* X, const GemmGeom& g, int r0, int kk,
                                 cudaStream_t s) {
    const size_t smem = (size_t)kAdjSB * (8 * NN + 2) * sizeof(c128);
    dim3 grid((unsigned)((g.N_m + kAdjPT - 1) / kAdjPT), (unsigned)g.n_f);
    if (g_adj_mt == 2) {
        auto k = gemm_adj_kernel<NN, 2>;
        cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        k<<<grid, 128, smem, s>>>(F, D, X, g, r0, kk);
    } else {
        auto k = gemm_adj_kernel<NN, 1>;
        cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        k<<<grid, 256, smem, s>>>(F, D, X, g, r0, kk);
    }
    return cudaGetLastError();
}

cudaError_t gemm_fwd_launch(int dt, const void* Fhat, const void* Xhat, void* partial, const GemmGeom& g,
                            cudaStream_t s) {
    if (dt == 0)
        return gemm32_umma_fwd_ok(g) ? gemm32_umma_fwd_launch(Fhat, Xhat, partial, g, s)
                                     : gemm32_fwd_launch(Fhat, Xhat, partial, g, s);
    const c128* F = static_cast<const c128*>(Fhat);
    const c128* X = static_cast<const c128*>(Xhat);
    c128* P = static_cast<c128*>(partial);
    for (int r0 = 0; r0 < g.k; r0 += 32) {
        const int kk = g.k - r0 < 32 ? g.k - r0 : 32;
        cudaError_t e = kk <= 8 ? fwd_launch_nn<1>(F, X, P, g, r0, kk, s)
                      : kk <= 16 ? fwd_launch_nn<2>(F, X, P, g, r0, kk, s)
                                 : fwd_launch_nn<4>(F, X, P, g, r0, kk, s);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

cudaError_t gemm_adj_launch(int dt, const void* Fhat, const void* Dhat, void* Xhat_out, const GemmGeom& g,
                            cudaStream_t s) {
    if (dt == 0)
        return gemm32_umma_adj_ok(g) ? gemm32_umma_adj_launch(Fhat, Dhat, Xhat_out, g, s)
                                     : gemm32_adj_launch(Fhat, Dhat, Xhat_out, g, s);
    const c128* F = static_cast<const c128*>(Fhat);
    const c128* D = static_cast<const c128*>(Dhat);
    c128* X = static_cast<c128*>(Xhat_out);
    for (int r0 = 0; r0 < g.k; r0 += 32) {
        const int kk = g.k - r0 < 32 ? g.k - r0 : 32;
        cudaError_t e = kk <= 8 ? adj_launch_nn<1>(F, D, X, g, r0, kk, s)
                      : kk <= 16 ? adj_launch_nn<2>(F, D, X, g, r0, kk, s)
                                 : adj_launch_nn<4>(F, D, X, g, r0, kk, s);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

}  // namespace tt
