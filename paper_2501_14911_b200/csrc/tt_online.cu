// tt_online.cu - the data-space side of the online phase behind the C ABI (include/tt.h, second half):
// tt_chol_* (K = L L^T, the two triangular solves of PAPER.md:294, 350), tt_assemble_K
// (K = Gamma_noise + F G*, column by column) and tt_map_* (the MAP point of
// eq 4.13).  F and G* are applied through the library's own tt_matvec / tt_rmatvec
// (FFT path, tt_api.cu); the triangular solves are the wavefront kernels of tt_trsv.cu; what is left
// here are a few element-wise data-space kernels and the sequencing.  No CPU fallback, no library BLAS.
#include <new>

#include "../../include/tt.h"
#include "tt_internal.h"

using namespace tt;

struct tt_chol {
    long long n = 0;
    int nblk = 0;
    double* Lt = nullptr;
    double* Dinv = nullptr;
    double* bt = nullptr;
    double* y = nullptr;
    double* xt = nullptr;
    unsigned* ticket = nullptr;
    size_t bytes = 0;
    mutable int last_cuda = 0;
};

struct tt_map {
    const tt_plan* F = nullptr;
    const tt_plan* G = nullptr;
    const tt_chol* K = nullptr;
    PlanInfo pi{};
    void* inv_nv = nullptr;   // [N_t*N_d] reals of the plans' dtype and layout: 1 / diag(Gamma_noise)
    void* yv = nullptr;       // Gamma_noise^{-1} d_obs
    void* dv = nullptr;       // F a, then z
    double* k64 = nullptr;    // [n] data-space vector in K's ordering, fp64 (rhs and solution of the K-solve)
    void* d_stage = nullptr;  // lazily: staging for tt_map_infer_host
    void* m_stage = nullptr;
    mutable int last_cuda = 0;
};

namespace tt {
long long chol_order(const ::tt_chol* c) { return c ? c->n : 0; }
}  // namespace tt

namespace {

inline size_t esize(int dtype) { return dtype == TT_F32 ? 4 : 8; }

template <typename H>
int fail_cuda(const H* h, cudaError_t e) {
    if (h) h->last_cuda = (int)e;
    (void)cudaGetLastError();
    return e == cudaErrorMemoryAllocation ? TT_ERR_OOM : TT_ERR_CUDA;
}

#define TTO_CUDA(h, call)                                  \
    do {                                                   \
        cudaError_t e__ = (call);                          \
        if (e__ != cudaSuccess) return fail_cuda(h, e__);  \
    } while (0)

bool is_device_ptr(const void* p) {
    cudaPointerAttributes attr;
    if (cudaPointerGetAttributes(&attr, p) != cudaSuccess) { (void)cudaGetLastError(); return false; }
    return attr.type == cudaMemoryTypeDevice || attr.type == cudaMemoryTypeManaged;
}

TrsvGeom geom(const tt_chol* c) {
    return TrsvGeom{c->n, c->nblk, c->Lt, c->Dinv, c->bt, c->y, c->xt, c->ticket};
}

// ---------------------------------------------------------------------------------------
// element-wise data-space kernels.  K's ordering is q = i*N_d + s; a data vector of a
// plan lives at  q  (TT_TIME_MAJOR)  or  s*N_t + i  (TT_SPACE_MAJOR).
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ long long lay(long long q, long long N_d, long long N_t, int layout) {
    if (layout == TT_TIME_MAJOR) return q;
    const long long i = q / N_d, s = q - i * N_d;
    return s * N_t + i;
}

template <typename T>
__global__ void recip_kernel(const T* __restrict__ nv, T* __restrict__ inv, long long n) {
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q < n) inv[q] = T(1) / nv[q];
}

// out = a * w, same layout on both sides (Gamma_noise^{-1} d_obs: diagonal)
template <typename T>
__global__ void mul_kernel(const T* __restrict__ a, const T* __restrict__ w, T* __restrict__ out, long long n) {
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q < n) out[q] = a[q] * w[q];
}

template <typename T>
__global__ void to_k_kernel(const T* __restrict__ v, double* __restrict__ k64, long long N_d, long long N_t, int layout) {
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q < N_d * N_t) k64[q] = (double)v[lay(q, N_d, N_t, layout)];
}

// z = y - c (y given) or z = c (y == nullptr), c in K's ordering and fp64, z and y in the plan's dtype and layout;
// the difference is formed in fp64 and rounded once.
template <typename T>
__global__ void from_k_kernel(const T* __restrict__ y, const double* __restrict__ k64, T* __restrict__ z, long long N_d,
                              long long N_t, int layout) {
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= N_d * N_t) return;
    const long long e = lay(q, N_d, N_t, layout);
    z[e] = y ? T((double)y[e] - k64[q]) : T(k64[q]);
}

// k-RHS data vectors: element (q, r) of D[.][.][k]
__device__ __forceinline__ long long lay_k(long long q, int r, long long N_d, long long N_t, int layout, int k) {
    if (layout == TT_TIME_MAJOR) return q * k + r;
    const long long i = q / N_d, s = q - i * N_d;
    return ((long long)r * N_d + s) * N_t + i;
}

// unit data vectors e_{col0}, ..., e_{col0+k-1} as the k columns of E (E zeroed beforehand)
template <typename T>
__global__ void unit_kernel(T* __restrict__ E, long long N_d, long long N_t, int layout, int k, long long col0) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r < k) E[lay_k(col0 + r, r, N_d, N_t, layout, k)] = T(1);
}

// K[q][col0 + r] = D[q][r] + (q == col0 + r ? noise_var[q] : 0)
template <typename T>
__global__ void scatter_K_kernel(const T* __restrict__ D, const T* __restrict__ nv, double* __restrict__ K, long long ldk,
                                 long long N_d, long long N_t, int layout, int k, long long col0) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= N_d * N_t * k) return;
    const long long q = t / k;
    const int r = (int)(t - q * k);
    double v = (double)D[lay_k(q, r, N_d, N_t, layout, k)];
    if (q == col0 + r) v += (double)nv[lay(q, N_d, N_t, layout)];
    K[(size_t)q * ldk + col0 + r] = v;
}

// out = u - out, element-wise over a parameter-sized vector (the subtraction of eq 4.7 / 4.8), grid-stride
template <typename T>
__global__ void __launch_bounds__(256) sub_from_kernel(const T* __restrict__ u, T* __restrict__ out, long long n) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) out[i] = u[i] - out[i];
}

inline unsigned nblocks(long long n, int t = 256) { return (unsigned)((n + t - 1) / t); }

bool same_shape(const PlanInfo& a, const PlanInfo& b) {
    return a.N_d == b.N_d && a.N_m == b.N_m && a.N_t == b.N_t && a.dtype == b.dtype && a.layout == b.layout &&
           a.dec == 1 && b.dec == 1;   // the online phase is defined on the data grid of F (N_t^d = N_t^m)
}

template <typename T>
int assemble_K_typed(const tt_plan* F, const tt_plan* G, const PlanInfo& pi, const T* nv, long long col0, long long ncols,
                     double* K, long long ldk, cudaStream_t s) {
    const long long n = pi.N_d * pi.N_t;
    const int kmax = pi.k_max;
    T *E = nullptr, *M = nullptr, *D = nullptr;
    cudaError_t e = cudaMalloc((void**)&E, (size_t)n * kmax * sizeof(T));
    if (e == cudaSuccess) e = cudaMalloc((void**)&D, (size_t)n * kmax * sizeof(T));
    if (e == cudaSuccess) e = cudaMalloc((void**)&M, (size_t)pi.N_t * pi.N_m * kmax * sizeof(T));
    int rc = TT_OK;
    if (e != cudaSuccess) { (void)cudaGetLastError(); rc = TT_ERR_OOM; }
    for (long long c0 = col0; rc == TT_OK && c0 < col0 + ncols; c0 += kmax) {
        const int k = (int)(col0 + ncols - c0 < kmax ? col0 + ncols - c0 : kmax);
        e = cudaMemsetAsync(E, 0, (size_t)n * k * sizeof(T), s);
        if (e != cudaSuccess) { (void)cudaGetLastError(); rc = TT_ERR_CUDA; break; }
        unit_kernel<T><<<nblocks(k, 64), 64, 0, s>>>(E, pi.N_d, pi.N_t, pi.layout, k, c0);
        rc = tt_rmatvec_batched(G, k, E, M, s);          // G* e_c
        if (rc == TT_OK) rc = tt_matvec_batched(F, k, M, D, s);  // F (G* e_c)
        if (rc != TT_OK) break;
        scatter_K_kernel<T><<<nblocks(n * k), 256, 0, s>>>(D, nv, K, ldk, pi.N_d, pi.N_t, pi.layout, k, c0);
        e = cudaGetLastError();
        if (e != cudaSuccess) { rc = TT_ERR_CUDA; break; }
    }
    e = cudaStreamSynchronize(s);
    if (e != cudaSuccess && rc == TT_OK) { (void)cudaGetLastError(); rc = TT_ERR_CUDA; }
    if (E) cudaFree(E);
    if (M) cudaFree(M);
    if (D) cudaFree(D);
    return rc;
}

// eq (4.13) in two halves, split where the N_m-sharded path has its one exchange step (the all-reduce of b = F a):
//   partial:  y = Gamma_noise^{-1} d_obs (kept in the tt_map),  a = G* y,  b = F a
//   finish :  c = K^{-1} b,  z = y - c,  m_map = G* z
template <typename T>
int map_partial_typed(const tt_map* m, const T* d_obs, T* a, T* b, cudaStream_t s) {
    const long long n = m->pi.N_d * m->pi.N_t;
    T* yv = static_cast<T*>(m->yv);
    mul_kernel<T><<<nblocks(n), 256, 0, s>>>(d_obs, static_cast<const T*>(m->inv_nv), yv, n);      // y = Gamma_noise^{-1} d_obs
    TTO_CUDA(m, cudaGetLastError());
    int rc;
    if ((rc = tt_rmatvec(m->G, yv, a, s)) != TT_OK) return rc;                                      // a = G* y
    return tt_matvec(m->F, a, b, s);                                                                // b = F a
}

template <typename T>
int map_finish_typed(const tt_map* m, const T* y /* nullptr: gain form, z = K^{-1} b */, const T* b, T* m_map,
                     cudaStream_t s, void* m_host = nullptr /* deliver m_map to host memory instead, copies pipelined */) {
    const PlanInfo& pi = m->pi;
    const long long n = pi.N_d * pi.N_t;
    T* dv = static_cast<T*>(m->dv);
    to_k_kernel<T><<<nblocks(n), 256, 0, s>>>(b, m->k64, pi.N_d, pi.N_t, pi.layout);
    int rc;
    if ((rc = tt_chol_solve(m->K, m->k64, m->k64, s)) != TT_OK) return rc;                          // c = K^{-1} b
    from_k_kernel<T><<<nblocks(n), 256, 0, s>>>(y, m->k64, dv, pi.N_d, pi.N_t, pi.layout);          // z = y - c  (or c)
    TTO_CUDA(m, cudaGetLastError());
    if (m_host) return plan_rmatvec_to_host(m->G, dv, m_host, s);
    return tt_rmatvec(m->G, dv, m_map, s);                                                          // m_map = G* z
}

// out = (I - G* K^{-1} F) u  (eq 4.7 with u = Gamma_prior v; eq 4.8 with u = m_prior), in the paper's order
template <typename T>
int smw_typed(const tt_map* m, const T* u, T* out, cudaStream_t s) {
    const PlanInfo& pi = m->pi;
    const long long n = pi.N_d * pi.N_t, nm = pi.N_m * pi.N_t;
    T* dv = static_cast<T*>(m->dv);
    int rc;
    if ((rc = tt_matvec(m->F, u, dv, s)) != TT_OK) return rc;                                       // b = F u
    to_k_kernel<T><<<nblocks(n), 256, 0, s>>>(dv, m->k64, pi.N_d, pi.N_t, pi.layout);
    if ((rc = tt_chol_solve(m->K, m->k64, m->k64, s)) != TT_OK) return rc;                          // c = K^{-1} b
    from_k_kernel<T><<<nblocks(n), 256, 0, s>>>(static_cast<const T*>(nullptr), m->k64, dv, pi.N_d, pi.N_t, pi.layout);
    if ((rc = tt_rmatvec(m->G, dv, out, s)) != TT_OK) return rc;                                    // e = G* c
    sub_from_kernel<T><<<148 * 8, 256, 0, s>>>(u, out, nm);                                        // out = u - e
    TTO_CUDA(m, cudaGetLastError());
    return TT_OK;
}

template <typename T>
int map_infer_typed(const tt_map* m, int form, const T* d_obs, T* m_map, cudaStream_t s, void* m_host = nullptr) {
    if (form == TT_MAP_GAIN) return map_finish_typed<T>(m, nullptr, d_obs, m_map, s, m_host);       // G* K^{-1} d_obs
    T* dv = static_cast<T*>(m->dv);
    const int rc = map_partial_typed<T>(m, d_obs, m_map, dv, s);                                    // a lives in m_map
    if (rc != TT_OK) return rc;
    return map_finish_typed<T>(m, static_cast<const T*>(m->yv), dv, m_map, s, m_host);
}

}  // namespace

extern "C" {

void tt_chol_destroy(tt_chol* c) {
    if (!c) return;
    void* bufs[] = {c->Lt, c->Dinv, c->bt, c->y, c->xt, c->ticket};
    for (void* b : bufs)
        if (b) cudaFree(b);
    delete c;
}

size_t tt_chol_device_bytes(const tt_chol* c) { return c ? c->bytes : 0; }
int tt_chol_last_cuda_error(const tt_chol* c) { return c ? c->last_cuda : 0; }

int tt_chol_create(tt_chol** out, int64_t n, const void* L, int64_t ld, void* stream) {
    if (!out) return TT_ERR_NULL;
    *out = nullptr;
    if (!L) return TT_ERR_NULL;
    if (n < 1 || ld < n || n > (int64_t)1 << 24) return TT_ERR_SHAPE;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { (void)cudaGetLastError(); return TT_ERR_NO_DEVICE; }
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        (void)cudaGetLastError();
        return TT_ERR_NO_DEVICE;
    }
    if (prop.major != 10) return TT_ERR_NO_DEVICE;

    tt_chol* c = new (std::nothrow) tt_chol();
    if (!c) return TT_ERR_OOM;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    constexpr long long NB = kTrsvNB;
    c->n = n;
    c->nblk = (int)((n + NB - 1) / NB);
    const size_t npad = (size_t)c->nblk * NB;
    const size_t lt_elems = (size_t)NB * NB * ((size_t)c->nblk * (size_t)(c->nblk - 1) / 2);
    int* bad = nullptr;
    double* slab = nullptr;
    int rc = TT_OK;
    auto alloc = [&](void** p, size_t bytes) -> bool {
        if (bytes == 0) bytes = 16;
        cudaError_t e = cudaMalloc(p, bytes);
        if (e != cudaSuccess) { *p = nullptr; rc = fail_cuda(c, e); return false; }
        c->bytes += bytes;
        return true;
    };
    auto bail = [&](int code) {
        if (bad) cudaFree(bad);
        if (slab) cudaFree(slab);
        tt_chol_destroy(c);
        return code;
    };
    if (!alloc((void**)&c->Lt, lt_elems * 8) || !alloc((void**)&c->Dinv, (size_t)c->nblk * NB * NB * 8) ||
        !alloc((void**)&c->bt, npad * 8) || !alloc((void**)&c->y, npad * 8) || !alloc((void**)&c->xt, npad * 8) ||
        !alloc((void**)&c->ticket, 16))
        return bail(rc);
    cudaError_t e = cudaMalloc((void**)&bad, sizeof(int));
    if (e == cudaSuccess) e = cudaMemsetAsync(bad, 0, sizeof(int), s);
    if (e != cudaSuccess) return bail(fail_cuda(c, e));

    if (is_device_ptr(L)) {
        e = trsv_prepare_launch(static_cast<const double*>(L), ld, 0, n, n, c->Dinv, c->Lt, bad, s);
        if (e != cudaSuccess) return bail(fail_cuda(c, e));
    } else {
        // host factor: block rows go through a device slab of <= 1 GiB (only columns <= last row of the slab are needed)
        long long rows = (long long)(((size_t)1 << 30) / ((size_t)n * 8));
        rows = rows / NB * NB;
        if (rows < NB) rows = NB;
        if (rows > (long long)npad) rows = (long long)npad;
        e = cudaMalloc((void**)&slab, (size_t)rows * (size_t)n * 8);
        if (e != cudaSuccess) return bail(fail_cuda(c, e));
        for (long long r0 = 0; r0 < n; r0 += rows) {
            const long long nr = n - r0 < rows ? n - r0 : rows;
            e = cudaMemcpy2DAsync(slab, (size_t)n * 8, static_cast<const double*>(L) + (size_t)r0 * ld, (size_t)ld * 8,
                                  (size_t)n * 8, (size_t)nr, cudaMemcpyHostToDevice, s);
            if (e == cudaSuccess) e = trsv_prepare_launch(slab, n, r0, nr, n, c->Dinv, c->Lt, bad, s);
            if (e == cudaSuccess) e = cudaStreamSynchronize(s);
            if (e != cudaSuccess) return bail(fail_cuda(c, e));
        }
    }
    int bad_h = 0;
    e = cudaMemcpyAsync(&bad_h, bad, sizeof(int), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return bail(fail_cuda(c, e));
    if (bad_h) return bail(TT_ERR_NOT_SPD);
    cudaFree(bad);
    if (slab) cudaFree(slab);
    *out = c;
    return TT_OK;
}

int tt_chol_solve(const tt_chol* c, const void* b, void* x, void* stream) {
    if (!c || !b || !x) return TT_ERR_NULL;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const TrsvGeom g = geom(c);
    TTO_CUDA(c, trsv_pre_launch(g, static_cast<const double*>(b), s));
    TTO_CUDA(c, trsv_fwd_launch(g, s));
    TTO_CUDA(c, trsv_bwd_launch(g, g.y, s));
    TTO_CUDA(c, trsv_post_launch(g, static_cast<double*>(x), s));
    return TT_OK;
}

int tt_chol_trsv(const tt_chol* c, int transposed, const void* b, void* x, void* stream) {
    if (!c || !b || !x) return TT_ERR_NULL;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const TrsvGeom g = geom(c);
    if (!transposed) {
        TTO_CUDA(c, trsv_pre_launch(g, static_cast<const double*>(b), s));
        TTO_CUDA(c, trsv_fwd_launch(g, s));
        TTO_CUDA(c, trsv_copy_launch(g.y, static_cast<double*>(x), c->n, s));
    } else {
        // bt doubles as the zero-padded copy of the right-hand side
        TTO_CUDA(c, trsv_pre_launch(g, nullptr, s));
        TTO_CUDA(c, cudaMemsetAsync(g.bt, 0, (size_t)c->nblk * kTrsvNB * 8, s));
        TTO_CUDA(c, trsv_copy_launch(static_cast<const double*>(b), g.bt, c->n, s));
        TTO_CUDA(c, trsv_bwd_launch(g, g.bt, s));
        TTO_CUDA(c, trsv_post_launch(g, static_cast<double*>(x), s));
    }
    return TT_OK;
}

int tt_assemble_K(const tt_plan* F, const tt_plan* G, const void* noise_var, int64_t col0, int64_t ncols, void* K,
                  int64_t ldk, void* stream) {
    if (!F || !G || !noise_var || !K) return TT_ERR_NULL;
    const PlanInfo pf = plan_info(F), pg = plan_info(G);
    if (!same_shape(pf, pg)) return TT_ERR_MISMATCH;
    const long long n = pf.N_d * pf.N_t;
    if (col0 < 0 || ncols < 0 || col0 + ncols > n || ldk < n) return TT_ERR_SHAPE;
    if (ncols == 0) return TT_OK;
    PlanInfo pi = pf;
    pi.k_max = pf.k_max < pg.k_max ? pf.k_max : pg.k_max;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (pi.dtype == TT_F32)
        return assemble_K_typed<float>(F, G, pi, static_cast<const float*>(noise_var), col0, ncols,
                                       static_cast<double*>(K), ldk, s);
    return assemble_K_typed<double>(F, G, pi, static_cast<const double*>(noise_var), col0, ncols,
                                    static_cast<double*>(K), ldk, s);
}

void tt_map_destroy(tt_map* m) {
    if (!m) return;
    void* bufs[] = {m->inv_nv, m->yv, m->dv, m->k64, m->d_stage, m->m_stage};
    for (void* b : bufs)
        if (b) cudaFree(b);
    delete m;
}

int tt_map_create(tt_map** out, const tt_plan* F, const tt_plan* G, const tt_chol* K, const void* noise_var,
                  void* stream) {
    if (!out) return TT_ERR_NULL;
    *out = nullptr;
    if (!G || !K || !noise_var) return TT_ERR_NULL;
    const PlanInfo pg = plan_info(G);
    if (F && !same_shape(plan_info(F), pg)) return TT_ERR_MISMATCH;
    const long long n = pg.N_d * pg.N_t;
    if (K->n != n || pg.dec != 1) return TT_ERR_MISMATCH;
    tt_map* m = new (std::nothrow) tt_map();
    if (!m) return TT_ERR_OOM;
    m->F = F; m->G = G; m->K = K; m->pi = pg;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const size_t es = esize(pg.dtype);
    cudaError_t e = cudaMalloc(&m->inv_nv, (size_t)n * es);
    if (e == cudaSuccess) e = cudaMalloc(&m->yv, (size_t)n * es);
    if (e == cudaSuccess) e = cudaMalloc(&m->dv, (size_t)n * es);
    if (e == cudaSuccess) e = cudaMalloc((void**)&m->k64, (size_t)n * 8);
    if (e == cudaSuccess) {
        if (pg.dtype == TT_F32)
            recip_kernel<float><<<nblocks(n), 256, 0, s>>>(static_cast<const float*>(noise_var),
                                                           static_cast<float*>(m->inv_nv), n);
        else
            recip_kernel<double><<<nblocks(n), 256, 0, s>>>(static_cast<const double*>(noise_var),
                                                            static_cast<double*>(m->inv_nv), n);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) {
        const int rc = fail_cuda(m, e);
        tt_map_destroy(m);
        return rc;
    }
    *out = m;
    return TT_OK;
}

int tt_map_infer(const tt_map* m, int form, const void* d_obs, void* m_map, void* stream) {
    if (!m || !d_obs || !m_map) return TT_ERR_NULL;
    if (form != TT_MAP_PAPER && form != TT_MAP_GAIN) return TT_ERR_SHAPE;
    if (form == TT_MAP_PAPER && !m->F) return TT_ERR_NULL;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (m->pi.dtype == TT_F32)
        return map_infer_typed<float>(m, form, static_cast<const float*>(d_obs), static_cast<float*>(m_map), s);
    return map_infer_typed<double>(m, form, static_cast<const double*>(d_obs), static_cast<double*>(m_map), s);
}

int tt_smw_apply(const tt_map* m, const void* u, void* out, void* stream) {
    if (!m || !u || !out || !m->F) return TT_ERR_NULL;
    if (u == out) return TT_ERR_ALIAS;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (m->pi.dtype == TT_F32) return smw_typed<float>(m, static_cast<const float*>(u), static_cast<float*>(out), s);
    return smw_typed<double>(m, static_cast<const double*>(u), static_cast<double*>(out), s);
}

// Phase 3 as compositions of the calls above with the p2q plans (tt_plan_create_coarse):
//   Gamma_post(q) v = F_q (I - G* K^{-1} F) G_q* v  (eq 4.10);   q_map = F_q m_map(d_obs) = Q d_obs  (eq 4.11, 4.14)
namespace {
bool q_plans_fit(const tt_map* m, const tt_plan* Fq, const tt_plan* Gq) {
    const PlanInfo a = plan_info(Fq);
    if (a.N_m != m->pi.N_m || a.N_t != m->pi.N_t || a.dtype != m->pi.dtype || a.layout != m->pi.layout) return false;
    if (!Gq) return true;
    const PlanInfo b = plan_info(Gq);
    return b.N_d == a.N_d && b.N_m == a.N_m && b.N_t == a.N_t && b.dtype == a.dtype && b.layout == a.layout && b.dec == a.dec;
}
}  // namespace

int tt_postcov_q_apply(const tt_map* m, const tt_plan* Fq, const tt_plan* Gq, const void* v, void* work, void* out,
                       void* stream) {
    if (!m || !Fq || !Gq || !v || !work || !out || !m->F) return TT_ERR_NULL;
    if (!q_plans_fit(m, Fq, Gq)) return TT_ERR_MISMATCH;
    const size_t nm = (size_t)m->pi.N_m * m->pi.N_t * esize(m->pi.dtype);
    void* a = work;
    void* u = static_cast<char*>(work) + nm;
    int rc;
    if ((rc = tt_rmatvec(Gq, v, a, stream)) != TT_OK) return rc;      // a = G_q* v
    if ((rc = tt_smw_apply(m, a, u, stream)) != TT_OK) return rc;     // u = (I - G* K^{-1} F) a
    return tt_matvec(Fq, u, out, stream);                             // F_q u
}

int tt_d2q_apply(const tt_map* m, const tt_plan* Fq, int form, const void* d_obs, void* work, void* q, void* stream) {
    if (!m || !Fq || !d_obs || !work || !q) return TT_ERR_NULL;
    if (!q_plans_fit(m, Fq, nullptr)) return TT_ERR_MISMATCH;
    const int rc = tt_map_infer(m, form, d_obs, work, stream);        // m_map
    if (rc != TT_OK) return rc;
    return tt_matvec(Fq, work, q, stream);                            // q_map = F_q m_map
}

int tt_map_infer_partial(const tt_map* m, const void* d_obs, void* a_scratch, void* b, void* stream) {
    if (!m || !d_obs || !a_scratch || !b || !m->F) return TT_ERR_NULL;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (m->pi.dtype == TT_F32)
        return map_partial_typed<float>(m, static_cast<const float*>(d_obs), static_cast<float*>(a_scratch),
                                        static_cast<float*>(b), s);
    return map_partial_typed<double>(m, static_cast<const double*>(d_obs), static_cast<double*>(a_scratch),
                                     static_cast<double*>(b), s);
}

int tt_map_infer_finish(const tt_map* m, const void* b, void* m_map, void* stream) {
    if (!m || !b || !m_map) return TT_ERR_NULL;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (m->pi.dtype == TT_F32)
        return map_finish_typed<float>(m, static_cast<const float*>(m->yv), static_cast<const float*>(b),
                                       static_cast<float*>(m_map), s);
    return map_finish_typed<double>(m, static_cast<const double*>(m->yv), static_cast<const double*>(b),
                                    static_cast<double*>(m_map), s);
}

int tt_map_infer_host(const tt_map* cm, int form, const void* d_obs_host, void* m_map_host, void* stream) {
    if (!cm || !d_obs_host || !m_map_host) return TT_ERR_NULL;
    if (form != TT_MAP_PAPER && form != TT_MAP_GAIN) return TT_ERR_SHAPE;
    if (form == TT_MAP_PAPER && !cm->F) return TT_ERR_NULL;
    tt_map* m = const_cast<tt_map*>(cm);
    const size_t es = esize(m->pi.dtype);
    const size_t nd = (size_t)m->pi.N_d * m->pi.N_t * es, nm = (size_t)m->pi.N_m * m->pi.N_t * es;
    if (!m->d_stage) TTO_CUDA(m, cudaMalloc(&m->d_stage, nd));
    if (form == TT_MAP_PAPER && !m->m_stage) TTO_CUDA(m, cudaMalloc(&m->m_stage, nm));   // a = G* y lives here
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    TTO_CUDA(m, cudaMemcpyAsync(m->d_stage, d_obs_host, nd, cudaMemcpyHostToDevice, s));
    // the final G* action delivers m_map range by range to the host while the next range computes
    if (m->pi.dtype == TT_F32)
        return map_infer_typed<float>(m, form, static_cast<const float*>(m->d_stage), static_cast<float*>(m->m_stage), s,
                                      m_map_host);
    return map_infer_typed<double>(m, form, static_cast<const double*>(m->d_stage), static_cast<double*>(m->m_stage), s,
                                   m_map_host);
}

}  // extern "C"
