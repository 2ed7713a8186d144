// plic_packed.cuh -- two cells per instruction: packed fp32x2 arithmetic (sm_100a).
//
// Blackwell adds add/mul/fma on a pair of fp32 values held in one 64-bit register pair
// (PTX add.f32x2 / mul.f32x2 / fma.rn.f32x2, SASS FADD2 / FMUL2 / FFMA2).  One issue slot then
// carries the arithmetic of two cells.  The PLIC kernels are bound by instruction issue, not
// by a single pipe (profiles/r01_ncu_summary.md: issue-active 78 %, fma 46 %, alu 44 %, xu
// 35 %), and about half of their instructions are plain mul/add/fma, so the branch-free
// variants run on pairs: every mul/add/fma is packed, while min/max/compare/select and the
// SFU ops, which have no packed form, are issued per half.
//
// F2 is a plain pair of floats.  mov.b64 {lo,hi} in the helpers only names the register
// pair; ptxas allocates both halves adjacent and emits no move for it.
#pragma once
#include "plic_math.cuh"

namespace plic {

struct F2 {
    float x, y;
};

__device__ __forceinline__ unsigned long long f2_pack(F2 a) {
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a.x), "f"(a.y));
    return r;
}
__device__ __forceinline__ F2 f2_unpack(unsigned long long r) {
    F2 a;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(a.x), "=f"(a.y) : "l"(r));
    return a;
}
__device__ __forceinline__ F2 f2(float k) { return F2{k, k}; }

__device__ __forceinline__ F2 fma2(F2 a, F2 b, F2 c) {
    unsigned long long r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(f2_pack(a)), "l"(f2_pack(b)), "l"(f2_pack(c)));
    return f2_unpack(r);
}
__device__ __forceinline__ F2 mul2(F2 a, F2 b) {
    unsigned long long r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(f2_pack(a)), "l"(f2_pack(b)));
    return f2_unpack(r);
}
__device__ __forceinline__ F2 add2(F2 a, F2 b) {
    unsigned long long r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(f2_pack(a)), "l"(f2_pack(b)));
    return f2_unpack(r);
}
// a - b as fma(b, -1, a): exact, one FFMA2 (the packed add has no negate modifier in PTX)
__device__ __forceinline__ F2 sub2(F2 a, F2 b) { return fma2(b, f2(-1.0f), a); }
__device__ __forceinline__ F2 mul2(F2 a, float k) { return mul2(a, f2(k)); }
__device__ __forceinline__ F2 fma2(F2 a, float k, F2 c) { return fma2(a, f2(k), c); }

// per-half operations (no packed form exists)
__device__ __forceinline__ F2 max2(F2 a, F2 b) { return F2{fmaxf(a.x, b.x), fmaxf(a.y, b.y)}; }
__device__ __forceinline__ F2 min2(F2 a, F2 b) { return F2{fminf(a.x, b.x), fminf(a.y, b.y)}; }
__device__ __forceinline__ F2 max2(F2 a, float k) { return F2{fmaxf(a.x, k), fmaxf(a.y, k)}; }

struct B2 {
    bool x, y;
};
__device__ __forceinline__ F2 sel2(B2 c, F2 a, F2 b) { return F2{c.x ? a.x : b.x, c.y ? a.y : b.y}; }
__device__ __forceinline__ B2 lt2(F2 a, F2 b) { return B2{a.x < b.x, a.y < b.y}; }
__device__ __forceinline__ B2 le2(F2 a, F2 b) { return B2{a.x <= b.x, a.y <= b.y}; }
__device__ __forceinline__ B2 gt2(F2 a, F2 b) { return B2{a.x > b.x, a.y > b.y}; }
__device__ __forceinline__ B2 and2(B2 a, B2 b) { return B2{a.x && b.x, a.y && b.y}; }
__device__ __forceinline__ B2 andnot2(B2 a, B2 b) { return B2{a.x && !b.x, a.y && !b.y}; }

__device__ __forceinline__ F2 rsqrt2(F2 a) { return F2{mufu_rsqrt(a.x), mufu_rsqrt(a.y)}; }
__device__ __forceinline__ F2 sqrt2(F2 a) { return F2{mufu_sqrt(a.x), mufu_sqrt(a.y)}; }
__device__ __forceinline__ F2 rcp2(F2 a) { return F2{mufu_rcp(a.x), mufu_rcp(a.y)}; }
__device__ __forceinline__ F2 lg2_2(F2 a) { return F2{mufu_lg2(a.x), mufu_lg2(a.y)}; }
__device__ __forceinline__ F2 ex2_2(F2 a) { return F2{mufu_ex2(a.x), mufu_ex2(a.y)}; }

// -sin(asin(C)/3), both halves: sin_third_asin_fast() of plic_math.cuh on a pair, negated
// (the Newton step's denominator is taken with the opposite sign, which costs nothing)
__device__ __forceinline__ F2 neg_sin_third_asin_fast2(F2 C) {
    const F2 C2 = mul2(C, C);
    F2 g = fma2(C2, f2(0.100619423f), f2(-0.0602495379f));
    g = fma2(g, C2, f2(0.073419422f));
    g = fma2(g, C2, f2(0.331531124f));
    g = mul2(g, C);
    const F2 g2 = mul2(g, g);
    const F2 num = fma2(mul2(g2, -8.0f), g, C);
    const F2 den = fma2(g2, 12.0f, f2(-3.0f));
    return mul2(num, rcp2(den));
}

// ---------------------------------------------------------------------------------------
// analytic inverse (eq. (25)/(26)), PLIC_FAST, for two cells at once.  Same arithmetic as
// Solver<ANALYTIC, true> was in round 1 -- every closed form evaluated and merged by select,
// (3)/(4) chosen a priori and served by one trigonometric evaluation -- but with no branch
// at all, so that the two cells of a pair (and the 32 lanes of a warp) share one instruction
// stream.  With R = 8 q (case 3) or u (case 4) and rho = rsqrt(R):
//   (3): d = n12 - sqrt(R) g(C),  C = (3/2) z rho           [2 sqrt(2q) = sqrt(8q)]
//   (4): d = S/2 - sqrt(R) g(C),  C = 6 q (n3 - W) rho^3
// Both roots are >= n2, which serves as the common floor (it also replaces a NaN from
// R = 0, i.e. n1 n2 flushed to zero, where the bracket [n2, n12] is narrower than fp32).
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ F2 solve_pair_analytic_fast(F2 V0, F2 nx, F2 ny, F2 nz) {
    const F2 a = F2{fabsf(nx.x), fabsf(nx.y)}, b = F2{fabsf(ny.x), fabsf(ny.y)},
             c = F2{fabsf(nz.x), fabsf(nz.y)};
    const F2 n1 = F2{min3(a.x, b.x, c.x), min3(a.y, b.y, c.y)};                 // eq. (2)
    const F2 n3 = F2{max3(a.x, b.x, c.x), max3(a.y, b.y, c.y)};                 // eq. (3)
    const F2 n2 = max2(min2(a, b), min2(max2(a, b), c));                        // eq. (4)
    // eq. (5): V = min(V0, 1 - V0); 2V saturated to [0, 1] (V0 outside [0,1] acts as 0 / 1)
    const F2 V = min2(V0, fma2(V0, -1.0f, f2(1.0f)));
    const F2 V2 = F2{__saturatef(V.x + V.x), __saturatef(V.y + V.y)};
    const F2 n12 = add2(n1, n2);
    const F2 W = mul2(V2, n3);                                                  // 2 V n3
    const F2 Wn2 = mul2(W, n2);
    const F2 x = mul2(Wn2, 3.0f);                                               // 6 V n2 n3
    const F2 s1 = mul2(n1, n1);
    const F2 hS = mul2(add2(n12, n3), 0.5f);
    // (2) and (1)
    const F2 d2 = fma2(n1, 0.5f, sqrt2(max2(fma2(s1, -1.0f / 12.0f, Wn2), 0.0f)));
    const F2 d1 = ex2_2(mul2(lg2_2(mul2(x, n1)), 1.0f / 3.0f));
    F2 d = sel2(lt2(x, s1), d1, d2);
    // (3)/(4)
    const F2 q = mul2(n1, n2);
    const F2 e = sub2(n3, n12);
    const F2 z = sub2(n12, W);
    const F2 ee = mul2(e, e);
    const F2 h = fma2(fma2(q, -6.0f, ee), e, mul2(mul2(q, z), -3.0f));          // F3(e)
    const B2 c4 = B2{e.x < 0.0f && h.x > 0.0f, e.y < 0.0f && h.y > 0.0f};
    const F2 R = sel2(c4, fma2(q, 4.0f, mul2(ee, -1.0f)), mul2(q, 8.0f));
    const F2 rho = rsqrt2(R);
    const F2 K4 = mul2(mul2(mul2(q, 6.0f), sub2(n3, W)), mul2(rho, rho));
    const F2 C = mul2(sel2(c4, K4, mul2(z, 1.5f)), rho);
    const F2 ng = neg_sin_third_asin_fast2(C);
    const F2 d34 = max2(fma2(mul2(R, rho), ng, sel2(c4, hS, n12)), n2);         // floor; drops NaN
    d = sel2(gt2(x, fma2(mul2(n2, 3.0f), sub2(n2, n1), s1)), d34, d);
    d = sel2(le2(n12, W), mul2(add2(W, n12), 0.5f), d);                         // (5)
    d = min2(d, hS);
    const F2 r = sub2(hS, d);
    // eq. (8): the sign of V0 - 1/2 on r >= 0
    const F2 t = fma2(V0, -1.0f, f2(0.5f));
    return F2{__uint_as_float(__float_as_uint(r.x) | (~__float_as_uint(t.x) & 0x80000000u)),
              __uint_as_float(__float_as_uint(r.y) | (~__float_as_uint(t.y) & 0x80000000u))};
}

}  // namespace plic
