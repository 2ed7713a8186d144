// plic_math.cuh -- scalar fp32 device primitives for the PLIC kernels (sm_100a).
//
//   Math<false>  the precise kernels' roots and reciprocals: IEEE-rounded division and square
//                root, CUDA libm cbrtf/asinf/acosf/sinf/cosf
//   mufu_*       one SFU (MUFU) instruction each: rsqrt/sqrt/rcp/lg2/ex2/cos .approx.ftz,
//                used by the PLIC_FAST kernels (plic_packed.cuh)
//   min3, max3   3-input min/max (FMNMX3, new on sm_100) for the sorting network of eq. (2)-(4)
#pragma once
#include <cuda_runtime.h>

namespace plic {

__device__ __forceinline__ float min3(float a, float b, float c) {
    float r;
    asm("min.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));
    return r;
}
__device__ __forceinline__ float max3(float a, float b, float c) {
    float r;
    asm("max.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));
    return r;
}
__device__ __forceinline__ float mufu_rsqrt(float x) {
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float mufu_sqrt(float x) {
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float mufu_rcp(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float mufu_lg2(float x) {
    float r;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float mufu_ex2(float x) {
    float r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float mufu_cos(float x) {
    float r;
    asm("cos.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

template <bool FAST>
struct Math;

template <>
struct Math<false> {
    static __device__ __forceinline__ float sqrt(float x) { return sqrtf(x); }
    static __device__ __forceinline__ float div(float a, float b) { return a / b; }
    static __device__ __forceinline__ float cbrt(float x) { return cbrtf(x); }
    // sin(pi/6 - acos(C)/3) of eq. (12) written as sin(asin(C)/3)  (pi/2 - acos = asin)
    static __device__ __forceinline__ float sin_third_asin(float C) {
        return sinf(asinf(fminf(C, 1.0f)) * (1.0f / 3.0f));
    }
    static __device__ __forceinline__ float acos(float x) { return acosf(fminf(x, 1.0f)); }
    static __device__ __forceinline__ float cos(float x) { return cosf(x); }
};

}  // namespace plic
