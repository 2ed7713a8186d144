// plic_probe.cuh -- instruction-rate probes for the roofline denominators (measurement support).
//
// The compute-bound entry points (nested intervals, plic_roundtrip_error, the precise methods)
// are scored against an instruction-issue or pipe roofline.  The per-SM rates those rooflines rest
// on are not documented for sm_100a, so they are measured: each probe kernel runs one kind of
// instruction in 8 independent dependency chains per thread, 16 warps per SM sub-partition,
// with nothing else in the loop but the loop counter, and plic_pipe_probe() reports how many
// warp-instructions of that kind one launch executes.  Rate = that count / time.
//
//   PROBE_FFMA    scalar fp32 FMA                (FMA pipe, both halves)
//   PROBE_FFMA2   packed fp32x2 FMA              (two cells per instruction; the fast kernels)
//   PROBE_MUFU    SFU op (rsqrt.approx)          (XU pipe: sqrt, rsqrt, rcp, lg2, ex2, cos)
//   PROBE_FMNMX   fp32 min/max                   (ALU pipe: min/max, compare, select, logic)
//   PROBE_LOP3    32-bit logic op                (ALU pipe; the sign transfer of nested-fast)
//   PROBE_NESTED  the nested-fast halving step   (2 FFMA2 + 2 LOP3 + 1 FADD2 per pair)
//   PROBE_DFMA    fp64 FMA                       (the pipe that bounds plic_solve_f64)
#pragma once
#include "plic_packed.cuh"

namespace plic {

enum : int { PROBE_FFMA = 0, PROBE_FFMA2 = 1, PROBE_MUFU = 2, PROBE_FMNMX = 3, PROBE_LOP3 = 4, PROBE_NESTED = 5,
             PROBE_FFMA_LOP3 = 6, PROBE_FFMA2_LOP3 = 7, PROBE_MUFU_FFMA4 = 8, PROBE_FFMA_FMNMX = 9, PROBE_FSEL = 10,
             PROBE_NESTED_SCALAR = 11, PROBE_NESTED_HYBRID = 12, PROBE_FADD = 13, PROBE_FMUL = 14, PROBE_FADD2 = 15,
             PROBE_3FP_LOP3 = 16, PROBE_DFMA = 17, PROBE_COUNT = 18 };
constexpr int kProbeChains = 8;        // independent chains per thread
constexpr int kProbeUnroll = 8;        // instructions per chain per loop trip
constexpr int kProbeBlocksPerSm = 8;   // x 256 threads = 16 warps per sub-partition

template <int PIPE>
struct ProbeOp;
template <>
struct ProbeOp<PROBE_FFMA> {
    typedef float T;
    static constexpr int kInst = 1;
    static __device__ __forceinline__ void step(float &a, float x, float y) {
        asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(a) : "f"(x), "f"(y));
    }
};
template <>
struct ProbeOp<PROBE_FFMA2> {
    typedef unsigned long long T;
    static constexpr int kInst = 1;
    static __device__ __forceinline__ void step(unsigned long long &a, unsigned long long x, unsigned long long y) {
        asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(a) : "l"(x), "l"(y));
    }
};
template <>
struct ProbeOp<PROBE_MUFU> {
    typedef float T;
    static constexpr int kInst = 1;
    static __device__ __forceinline__ void step(float &a, float, float) {
        asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(a));
    }
};
template <>
struct ProbeOp<PROBE_FMNMX> {
    typedef float T;
    static constexpr int kInst = 2;
    static __device__ __forceinline__ void step(float &a, float x, float y) {
        asm volatile("max.f32 %0, %0, %1;\n\tmin.f32 %0, %0, %2;" : "+f"(a) : "f"(x), "f"(y));
    }
};
template <>
struct ProbeOp<PROBE_LOP3> {
    typedef unsigned T;
    static constexpr int kInst = 1;
    static __device__ __forceinline__ void step(unsigned &a, unsigned x, unsigned y) {
        asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a) : "r"(x), "r"(y));
    }
};

// mixes: does an ALU-pipe instruction overlap with an FMA-pipe or SFU instruction?
template <>
struct ProbeOp<PROBE_FFMA_LOP3> {
    typedef float T;
    static constexpr int kInst = 2;
    static __device__ __forceinline__ void step(float &a, float x, float y) {
        asm volatile("{ .reg .b32 t; fma.rn.f32 %0, %0, %1, %2; mov.b32 t, %0; lop3.b32 t, t, 0x007fffff, 0x3f800000, 0xEA; mov.b32 %0, t; }"
                     : "+f"(a) : "f"(x), "f"(y));
    }
};
template <>
struct ProbeOp<PROBE_FFMA2_LOP3> {
    typedef unsigned long long T;
    static constexpr int kInst = 2;
    static __device__ __forceinline__ void step(unsigned long long &a, unsigned long long x, unsigned long long y) {
        asm volatile("{ .reg .b32 lo, hi; fma.rn.f32x2 %0, %0, %1, %2; mov.b64 {lo, hi}, %0; lop3.b32 lo, lo, 0x007fffff, 0x3f800000, 0xEA; mov.b64 %0, {lo, hi}; }"
                     : "+l"(a) : "l"(x), "l"(y));
    }
};
template <>
struct ProbeOp<PROBE_MUFU_FFMA4> {
    typedef float T;
    static constexpr int kInst = 5;
    static __device__ __forceinline__ void step(float &a, float x, float y) {
        asm volatile("rsqrt.approx.ftz.f32 %0, %0;\n\tfma.rn.f32 %0, %0, %1, %2;\n\tfma.rn.f32 %0, %0, %1, %2;\n\t"
                     "fma.rn.f32 %0, %0, %1, %2;\n\tfma.rn.f32 %0, %0, %1, %2;" : "+f"(a) : "f"(x), "f"(y));
    }
};
template <>
struct ProbeOp<PROBE_FFMA_FMNMX> {
    typedef float T;
    static constexpr int kInst = 2;
    static __device__ __forceinline__ void step(float &a, float x, float y) {
        asm volatile("fma.rn.f32 %0, %0, %1, %2;\n\tmax.f32 %0, %0, %2;" : "+f"(a) : "f"(x), "f"(y));
    }
};
template <>
struct ProbeOp<PROBE_FSEL> {
    typedef float T;
    static constexpr int kInst = 2;
    static __device__ __forceinline__ void step(float &a, float x, float y) {
        asm volatile("{ .reg .pred p; setp.lt.f32 p, %0, %1; selp.f32 %0, %2, %0, p; }" : "+f"(a) : "f"(x), "f"(y));
    }
};

template <>
struct ProbeOp<PROBE_FADD> {
    typedef float T;
    static constexpr int kInst = 1;
    static __device__ __forceinline__ void step(float &a, float x, float y) {
        asm volatile("add.rn.f32 %0, %0, %2;" : "+f"(a) : "f"(x), "f"(y));
    }
};
template <>
struct ProbeOp<PROBE_FMUL> {
    typedef float T;
    static constexpr int kInst = 1;
    static __device__ __forceinline__ void step(float &a, float x, float y) {
        asm volatile("mul.rn.f32 %0, %0, %1;" : "+f"(a) : "f"(x), "f"(y));
    }
};
template <>
struct ProbeOp<PROBE_FADD2> {
    typedef unsigned long long T;
    static constexpr int kInst = 1;
    static __device__ __forceinline__ void step(unsigned long long &a, unsigned long long x, unsigned long long y) {
        asm volatile("add.rn.f32x2 %0, %0, %2;" : "+l"(a) : "l"(x), "l"(y));
    }
};
template <>
struct ProbeOp<PROBE_3FP_LOP3> {      // the scalar nested step's mix without its dependencies on the LOP3
    typedef float T;
    static constexpr int kInst = 4;
    static __device__ __forceinline__ void step(float &a, float x, float y) {
        asm volatile("{ .reg .b32 t; fma.rn.f32 %0, %0, %1, %2; fma.rn.f32 %0, %0, %1, %2; mov.b32 t, %0; "
                     "lop3.b32 t, t, 0x007fffff, 0x3f800000, 0xEA; mov.b32 %0, t; add.rn.f32 %0, %0, %2; }"
                     : "+f"(a) : "f"(x), "f"(y));
    }
};

template <int PIPE>
__global__ void __launch_bounds__(256)
pipe_probe(float *sink, int trips) {
    typedef typename ProbeOp<PIPE>::T T;
    T a[kProbeChains];
    const float seed = 1.0f + (float)threadIdx.x * (1.0f / 4096.0f);
    T x, y;
    if constexpr (sizeof(T) == 8) {
        x = f2_pack(F2{0.999f, 1.001f});
        y = f2_pack(F2{seed * 1e-3f, seed * 2e-3f});
        for (int j = 0; j < kProbeChains; ++j) a[j] = f2_pack(F2{seed + j, seed - j});
    } else if constexpr (PIPE == PROBE_LOP3) {
        x = threadIdx.x * 2654435761u;
        y = blockIdx.x * 40503u + 1u;
        for (int j = 0; j < kProbeChains; ++j) a[j] = threadIdx.x + 77u * j;
    } else {
        x = (PIPE == PROBE_FMNMX || PIPE == PROBE_FSEL) ? seed : 0.999f;
        y = (PIPE == PROBE_FMNMX || PIPE == PROBE_FSEL) ? seed + 3.0f : seed * 1e-3f;
        for (int j = 0; j < kProbeChains; ++j) a[j] = seed + (float)j;
    }
    for (int t = 0; t < trips; ++t) {
#pragma unroll
        for (int u = 0; u < kProbeUnroll; ++u)
#pragma unroll
            for (int j = 0; j < kProbeChains; ++j) ProbeOp<PIPE>::step(a[j], x, y);
    }
    float acc = 0.0f;
    for (int j = 0; j < kProbeChains; ++j) {
        if constexpr (sizeof(T) == 8) { const F2 v = f2_unpack(a[j]); acc += v.x + v.y; }
        else if constexpr (PIPE == PROBE_LOP3) acc += (float)(a[j] & 0xffu);
        else acc += a[j];
    }
    if (acc == 123456.789f) sink[threadIdx.x] = acc;      // never true: keeps the chains alive
}

// fp64 FMA in 8 independent chains per thread (kProbeChains x kProbeUnroll instructions per trip)
__global__ void __launch_bounds__(256)
pipe_probe_dfma(float *sink, int trips) {
    double a[kProbeChains];
    const double seed = 1.0 + (double)threadIdx.x * (1.0 / 4096.0);
    const double x = 0.999, y = seed * 1e-3;
    for (int j = 0; j < kProbeChains; ++j) a[j] = seed + (double)j;
    for (int t = 0; t < trips; ++t) {
#pragma unroll
        for (int u = 0; u < kProbeUnroll; ++u)
#pragma unroll
            for (int j = 0; j < kProbeChains; ++j) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(a[j]) : "d"(x), "d"(y));
    }
    double acc = 0.0;
    for (int j = 0; j < kProbeChains; ++j) acc += a[j];
    if (acc == 123456.789) sink[threadIdx.x] = (float)acc;
}

// the halving step of PairSolver<NESTED> on 4 independent pairs per thread
__global__ void __launch_bounds__(256)
pipe_probe_nested(float *sink, int trips) {
    const float seed = (float)threadIdx.x * (1.0f / 512.0f);
    F2 c[4], nP[4], nR[4];
    for (int j = 0; j < 4; ++j) {
        c[j] = F2{-0.5f - seed * 0.01f * j, -0.4f - seed * 0.02f};
        nP[j] = F2{-3.0f - seed, -2.5f + seed * 0.3f + j};
        nR[j] = F2{-0.7f - seed * 0.1f, -0.9f - 0.1f * j + seed};
    }
    const unsigned mask = sign_mask_register();
    for (int t = 0; t < trips; ++t) {
#pragma unroll
        for (int j = 0; j < 4; ++j) NestedSteps<0, 16>::run(c[j], nP[j], nR[j], mask);
    }
    float acc = 0.0f;
    for (int j = 0; j < 4; ++j) acc += c[j].x + c[j].y;
    if (acc == 123456.789f) sink[threadIdx.x] = acc;
}

// the same step with scalar arithmetic (VARIANT 0: FFMA, FFMA, LOP3, FADD per cell) or packed
// FMAs and scalar adds (VARIANT 1), on 8 cells per thread
template <int VARIANT>
__global__ void __launch_bounds__(256)
pipe_probe_nested_alt(float *sink, int trips) {
    const float seed = (float)threadIdx.x * (1.0f / 512.0f);
    float c[8], nP[8], nR[8];
    for (int j = 0; j < 8; ++j) {
        c[j] = -0.5f - seed * 0.01f * j;
        nP[j] = -3.0f - seed + 0.25f * j;
        nR[j] = -0.7f - seed * 0.1f - 0.05f * j;
    }
    const unsigned mask = sign_mask_register();
    for (int t = 0; t < trips; ++t) {
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            const unsigned step = (unsigned)(127 - (k + 2)) << 23;
#pragma unroll
            for (int j = 0; j < 8; j += 2) {
                float g0, g1;
                if (VARIANT == 0) {
                    g0 = fmaf(fmaf(c[j], c[j], nP[j]), c[j], nR[j]);
                    g1 = fmaf(fmaf(c[j + 1], c[j + 1], nP[j + 1]), c[j + 1], nR[j + 1]);
                } else {
                    const F2 cc{c[j], c[j + 1]};
                    const F2 G = fma2(fma2(cc, cc, F2{nP[j], nP[j + 1]}), cc, F2{nR[j], nR[j + 1]});
                    g0 = G.x; g1 = G.y;
                }
                unsigned r0, r1;
                asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=r"(r0) : "r"(__float_as_uint(g0)), "r"(mask), "r"(step));
                asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=r"(r1) : "r"(__float_as_uint(g1)), "r"(mask), "r"(step));
                c[j] += __uint_as_float(r0);
                c[j + 1] += __uint_as_float(r1);
            }
        }
    }
    float acc = 0.0f;
    for (int j = 0; j < 8; ++j) acc += c[j];
    if (acc == 123456.789f) sink[threadIdx.x] = acc;
}

}  // namespace plic
