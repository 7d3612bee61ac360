// dt_common.cuh -- shared device helpers for the DominoTree builder kernels (sm_100a).
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace dt {

constexpr int kWarp = 32;

// ---- element type helpers: T is __nv_bfloat16 or float -------------------------------------
template <typename T> struct ElemTraits;
template <> struct ElemTraits<__nv_bfloat16> {
    static constexpr int kVec = 8;              // elements per 16-byte vector
    static __device__ __forceinline__ float to_f32(__nv_bfloat16 v) { return __bfloat162float(v); }
};
template <> struct ElemTraits<float> {
    static constexpr int kVec = 4;
    static __device__ __forceinline__ float to_f32(float v) { return v; }
};

__device__ __forceinline__ float bf16_bits_to_f32(uint32_t hi16) { return __uint_as_float(hi16 << 16); }

// Unpack the 8 bf16 of a uint4 into floats (element 0 = lowest address).
__device__ __forceinline__ void unpack8(const uint4 &v, float (&f)[8]) {
    f[0] = __uint_as_float(v.x << 16); f[1] = __uint_as_float(v.x & 0xFFFF0000u);
    f[2] = __uint_as_float(v.y << 16); f[3] = __uint_as_float(v.y & 0xFFFF0000u);
    f[4] = __uint_as_float(v.z << 16); f[5] = __uint_as_float(v.z & 0xFFFF0000u);
    f[6] = __uint_as_float(v.w << 16); f[7] = __uint_as_float(v.w & 0xFFFF0000u);
}

// Order-preserving map float -> uint32 (larger float <=> larger key), with -0 folded onto +0 so
// that equal values give equal keys.  NaN is outside the contract (dominotree.h).
__device__ __forceinline__ uint32_t ord_key(float v) {
    uint32_t b = __float_as_uint(v);
    if (b == 0x80000000u) b = 0u;
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ float ord_key_inv(uint32_t k) {
    uint32_t b = (k & 0x80000000u) ? (k & 0x7FFFFFFFu) : ~k;
    return __uint_as_float(b);
}

// 128-bit streaming global load (read-once data: do not allocate in L1).
__device__ __forceinline__ uint4 ld_stream_v4(const void *p) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}
// 128-bit read-only load that may stay in L1/L2 (weights, reused rows).
__device__ __forceinline__ uint4 ld_ro_v4(const void *p) {
    return __ldg(reinterpret_cast<const uint4 *>(p));
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

__device__ __forceinline__ float sigmoidf_acc(float x) { return 1.0f / (1.0f + expf(-x)); }

// Fast gate functions for the fused expansion kernel: ex2.approx-based, relative error ~1e-6 -- two orders
// below the 1e-4 ordering margin.
__device__ __forceinline__ float sigmoidf_fast(float x) { return __fdividef(1.0f, 1.0f + __expf(-x)); }
__device__ __forceinline__ float tanhf_fast(float x) {
    const float xc = fminf(fmaxf(x, -15.f), 15.f);
    return 1.0f - __fdividef(2.0f, 1.0f + __expf(2.0f * xc));
}

// generic element load -> float
template <typename T> __device__ __forceinline__ float ldf(const T *p, size_t i) {
    return ElemTraits<T>::to_f32(p[i]);
}

__device__ __forceinline__ unsigned long long wave_timer() {
    unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t;
}
// In-kernel timeline of the persistent expansion kernels (measurement builds only: `python -m paper_2607_08642_b200.build --trace` compiles the separate
// libdominotree_trace.so with -DDT_TRACE, read by `bench.py --trace`): thread 0 of GRU CTA 0 (role 0) and of request
// CTA 0 (role 1) of dt_wave.cuh / dt_fused.cuh stamp %globaltimer at fixed points of the first kWvTraceSteps steps.
constexpr int kWvTraceSteps = 64, kWvTraceStamps = 16;
#ifdef DT_TRACE
__device__ unsigned long long g_wv_trace[2][kWvTraceSteps][kWvTraceStamps];
// one PREDICATED store by thread 0 (no branch: a thread-0-only branch would leave its warp diverged and slow every warp
// collective after it; no store at all by the other threads: a release fence waits for every store in flight)
#define WV_TR(role, cond, step, i) do { \
        const bool wv_on__ = (threadIdx.x == 0) && (cond) && (step) < kWvTraceSteps; \
        unsigned long long *wv_dst__ = &g_wv_trace[role][wv_on__ ? (step) : 0][i]; \
        const unsigned long long wv_t__ = wave_timer(); \
        asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %2, 0;\n\t@p st.global.u64 [%0], %1;\n\t}\n" \
                     :: "l"(wv_dst__), "l"(wv_t__), "r"((unsigned int)wv_on__) : "memory"); } while (0)
#define WV_TRT(tt, role, cond, step, i) do { \
        const bool wv_on__ = (threadIdx.x == (tt)) && (cond) && (step) < kWvTraceSteps; \
        unsigned long long *wv_dst__ = &g_wv_trace[role][wv_on__ ? (step) : 0][i]; \
        const unsigned long long wv_t__ = wave_timer(); \
        asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %2, 0;\n\t@p st.global.u64 [%0], %1;\n\t}\n" \
                     :: "l"(wv_dst__), "l"(wv_t__), "r"((unsigned int)wv_on__) : "memory"); } while (0)
#else
#define WV_TR(role, cond, step, i) do { } while (0)
#define WV_TRT(tt, role, cond, step, i) do { } while (0)
#endif

}  // namespace dt
