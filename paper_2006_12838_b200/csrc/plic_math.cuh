// plic_math.cuh -- scalar fp32 device primitives for the PLIC kernels (sm_100a).
//
// Two flavours of every root / reciprocal, selected at compile time:
//   Math<false>  IEEE-rounded division and square root, CUDA libm cbrtf/asinf/acosf/sinf/cosf
//   Math<true>   one SFU (MUFU) instruction each: rsqrt/sqrt/rcp/lg2/ex2/cos .approx.ftz
// plus 3-input min/max (FMNMX3, new on sm_100) for the sorting network of eq. (2)-(4).
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

// sin(asin(C)/3) for C in [0, 0.9]: the root g in [0, 0.36] of the triple-angle relation
// 3g - 4g^3 = C.  An odd minimax start value C*P3(C^2) (|err| < 2.0e-4 on [0, 0.9]) is
// polished by one Newton step g <- (C - 8g^3)/(3 - 12g^2), whose denominator stays >= 1.4;
// the result is within 1.3e-7 of the exact value.  This replaces the asin + sin pair of the
// trigonometric cubic root (eq. (12)) in the PLIC_FAST kernels: the argument
// range C <= 5/(4 sqrt 2) = 0.884 is a property of cases (3)/(4) ("trig range").
// Coefficients: fit_coefficients.py.
__device__ __forceinline__ float sin_third_asin_fast(float C) {
    const float C2 = C * C;
    float g = fmaf(C2, 0.100619423f, -0.0602495379f);
    g = fmaf(g, C2, 0.073419422f);
    g = fmaf(g, C2, 0.331531124f);
    g *= C;
    const float g2 = g * g;
    const float num = fmaf(-8.0f * g2, g, C);
    const float den = fmaf(-12.0f, g2, 3.0f);
    return num * mufu_rcp(den);
}

// acos(x) for x in [0, 1] as sqrt(1-x) * Q5(x), |err| < 1.2e-6 (minimax fit,
// fit_coefficients.py).  Used by the PLIC_FAST SZ kernel, where the angle is divided by 3.
__device__ __forceinline__ float acos_fast(float x) {
    float p = fmaf(x, -0.004337173733f, 0.01934827404f);
    p = fmaf(p, x, -0.04495724702f);
    p = fmaf(p, x, 0.08787565452f);
    p = fmaf(p, x, -0.2145122723f);
    p = fmaf(p, x, 1.570795206f);
    return mufu_sqrt(fmaxf(1.0f - x, 0.0f)) * p;
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

template <>
struct Math<true> {
    static __device__ __forceinline__ float sqrt(float x) { return mufu_sqrt(x); }
    static __device__ __forceinline__ float div(float a, float b) { return a * mufu_rcp(b); }
    // exp2(log2(x)/3); lg2(0) = -inf -> ex2 = 0.  Relative error < 1e-6 on the range used.
    static __device__ __forceinline__ float cbrt(float x) {
        return mufu_ex2(mufu_lg2(x) * (1.0f / 3.0f));
    }
    static __device__ __forceinline__ float sin_third_asin(float C) {
        return sin_third_asin_fast(C);
    }
    static __device__ __forceinline__ float acos(float x) { return acos_fast(fminf(x, 1.0f)); }
    static __device__ __forceinline__ float cos(float x) { return mufu_cos(x); }
};

}  // namespace plic
