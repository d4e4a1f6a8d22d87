// tt_common.cuh - small device-side vocabulary shared by the libtt kernels (sm_100a).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tt {

// Interleaved complex number, aligned so that one element is one 64-/128-bit access.
template <typename R>
struct alignas(2 * sizeof(R)) Cx {
    R re, im;
};
using c64 = Cx<float>;
using c128 = Cx<double>;

template <typename R> __host__ __device__ __forceinline__ Cx<R> mk(R a, R b) { Cx<R> z; z.re = a; z.im = b; return z; }
template <typename R> __device__ __forceinline__ Cx<R> operator+(Cx<R> a, Cx<R> b) { return mk<R>(a.re + b.re, a.im + b.im); }
template <typename R> __device__ __forceinline__ Cx<R> operator-(Cx<R> a, Cx<R> b) { return mk<R>(a.re - b.re, a.im - b.im); }
template <typename R> __device__ __forceinline__ Cx<R> operator*(Cx<R> a, Cx<R> b) {
    return mk<R>(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re);
}
template <typename R> __device__ __forceinline__ Cx<R> conj(Cx<R> a) { return mk<R>(a.re, -a.im); }
// a * (-i)  and  a * (+i)
template <typename R> __device__ __forceinline__ Cx<R> mul_mi(Cx<R> a) { return mk<R>(a.im, -a.re); }
template <typename R> __device__ __forceinline__ Cx<R> mul_pi(Cx<R> a) { return mk<R>(-a.im, a.re); }
// acc += a * b
template <typename R> __device__ __forceinline__ void cmac(Cx<R>& acc, Cx<R> a, Cx<R> b) {
    acc.re = fma(a.re, b.re, acc.re); acc.re = fma(-a.im, b.im, acc.re);
    acc.im = fma(a.re, b.im, acc.im); acc.im = fma(a.im, b.re, acc.im);
}
// acc += conj(a) * b
template <typename R> __device__ __forceinline__ void cmac_conj(Cx<R>& acc, Cx<R> a, Cx<R> b) {
    acc.re = fma(a.re, b.re, acc.re); acc.re = fma(a.im, b.im, acc.re);
    acc.im = fma(a.re, b.im, acc.im); acc.im = fma(-a.im, b.re, acc.im);
}

// 128-bit streaming loads of data that is read exactly once (Fhat): read-only path,
// no L1 allocation, so that the stream does not push the staged spectrum out of L1.
__device__ __forceinline__ float4 ldg_stream(const float4* p) {
    float4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}
__device__ __forceinline__ double2 ldg_stream(const double2* p) {
    double2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0,%1}, [%2];"
                 : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}

// L2 eviction policies (createpolicy) for two kernels that hand an intermediate over THROUGH the L2: the one-pass stream
// is marked evict-first, the intermediate evict-last, and the consumer reads it past L1 and drops its lines without a write-back.
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ uint64_t l2_policy_evict_last() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ float4 ldg_stream(const float4* p, uint64_t pol) {
    float4 v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.f32 {%0,%1,%2,%3}, [%4], %5;"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ double2 ldg_stream(const double2* p, uint64_t pol) {
    double2 v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;"
                 : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ void stg_hint(float4* p, float4 v, uint64_t pol) {
    asm volatile("st.global.L2::cache_hint.v4.f32 [%0], {%1,%2,%3,%4}, %5;" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w), "l"(pol) : "memory");
}
__device__ __forceinline__ void stg_hint(double2* p, double2 v, uint64_t pol) {
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1,%2}, %3;" ::"l"(p), "d"(v.x), "d"(v.y), "l"(pol) : "memory");
}
__device__ __forceinline__ Cx<float> ld_cg(const Cx<float>* p) {
    Cx<float> v;
    asm volatile("ld.global.cg.v2.f32 {%0,%1}, [%2];" : "=f"(v.re), "=f"(v.im) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ Cx<double> ld_cg(const Cx<double>* p) {
    Cx<double> v;
    asm volatile("ld.global.cg.v2.f64 {%0,%1}, [%2];" : "=d"(v.re), "=d"(v.im) : "l"(p) : "memory");
    return v;
}
// The 128-byte line at p (128-byte aligned) will not be read again before it is overwritten: drop it from the L2 without
// writing it back to HBM.
__device__ __forceinline__ void l2_discard_line(const void* p) {
    asm volatile("discard.global.L2 [%0], 128;" ::"l"(p) : "memory");
}

// cp.async (LDGSTS): global -> shared without a register stage.  `valid` false: the destination is zero-filled (src-size 0).
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc, bool valid) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    const int n = valid ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(d), "l"(gsrc), "r"(n) : "memory");
}
__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gsrc, bool valid) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    const int n = valid ? 8 : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(d), "l"(gsrc), "r"(n) : "memory");
}
__device__ __forceinline__ void cp_async4(void* smem_dst, const void* gsrc, bool valid) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    const int n = valid ? 4 : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(d), "l"(gsrc), "r"(n) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// 16-byte vector of complex numbers: 2 x complex64 or 1 x complex128.
template <typename R> struct Vec16;
template <> struct Vec16<float> {
    using type = float4;
    static constexpr int n = 2;
    static __device__ __forceinline__ c64 get(const float4& v, int i) { return i == 0 ? mk<float>(v.x, v.y) : mk<float>(v.z, v.w); }
    static __device__ __forceinline__ float4 zero() { return make_float4(0.f, 0.f, 0.f, 0.f); }
    static __device__ __forceinline__ float4 pack(c64 a, c64 b) { return make_float4(a.re, a.im, b.re, b.im); }
};
template <> struct Vec16<double> {
    using type = double2;
    static constexpr int n = 1;
    static __device__ __forceinline__ c128 get(const double2& v, int) { return mk<double>(v.x, v.y); }
    static __device__ __forceinline__ double2 zero() { return make_double2(0.0, 0.0); }
    static __device__ __forceinline__ double2 pack(c128 a, c128) { return make_double2(a.re, a.im); }
};

template <typename R> __device__ __forceinline__ Cx<R> warp_sum(Cx<R> v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        v.re += __shfl_xor_sync(0xffffffffu, v.re, o);
        v.im += __shfl_xor_sync(0xffffffffu, v.im, o);
    }
    return v;
}

}  // namespace tt
