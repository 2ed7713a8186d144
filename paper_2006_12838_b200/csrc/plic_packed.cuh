// plic_packed.cuh -- two cells per instruction: packed fp32x2 arithmetic (sm_100a).
//
// Blackwell adds add/mul/fma on a pair of fp32 values held in one 64-bit register pair
// (PTX add.f32x2 / mul.f32x2 / fma.rn.f32x2, SASS FADD2 / FMUL2 / FFMA2).  About half the
// instructions of a branch-free PLIC method are plain mul/add/fma, so the PLIC_FAST variants run
// on pairs: every mul/add/fma is packed, while min/max/compare/select and the SFU ops, which
// have no packed form, are issued per half.  A packed instruction halves the instruction count
// of that arithmetic but holds the issue port for two clocks (plic_probe.cuh: FFMA2 0.50 per
// clock, FFMA2 + LOP3 0.66 = three clocks per pair), so the ceiling of these kernels is counted
// in issue slots = instructions + packed instructions; what packing buys
// is registers, instruction-cache and scoreboard pressure.
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

// -sin(asin(C)/3) (TWICE: -2 sin(asin(C)/3)) for C in [0, 0.9], both halves.  g = sin(asin(C)/3) is the
// root in [0, 0.36] of the triple-angle relation 3g - 4g^3 = C.  An odd minimax start value C*P3(C^2)
// (|err| < 2.0e-4 on [0, 0.9]) is polished by one Newton step g <- (C - 8g^3)/(3 - 12g^2),
// whose denominator stays >= 1.4; the result is within 1.3e-7 of the exact value.  This
// replaces the asin + sin pair of the trigonometric cubic root (eq. (12)): the
// argument range C <= 5/(4 sqrt 2) = 0.884 is a property of cases (3)/(4) ("trig
// range").  The step's denominator is taken with the opposite sign (and halved for TWICE), which
// negates (doubles) the result at no cost.  Coefficients: fit_coefficients.py.
template <bool TWICE>
__device__ __forceinline__ F2 neg_sin_third_asin_fast2(F2 C) {
    const F2 C2 = mul2(C, C);
    F2 g = fma2(C2, f2(0.100619423f), f2(-0.0602495379f));
    g = fma2(g, C2, f2(0.073419422f));
    g = fma2(g, C2, f2(0.331531124f));
    g = mul2(g, C);
    const F2 g2 = mul2(g, g);
    const F2 num = fma2(mul2(g2, -8.0f), g, C);
    const F2 den = TWICE ? fma2(g2, 6.0f, f2(-1.5f)) : fma2(g2, 12.0f, f2(-3.0f));
    return mul2(num, rcp2(den));
}

__device__ __forceinline__ F2 cos2(F2 a) { return F2{mufu_cos(a.x), mufu_cos(a.y)}; }
__device__ __forceinline__ F2 sat2(F2 a) { return F2{__saturatef(a.x), __saturatef(a.y)}; }
__device__ __forceinline__ F2 abs2(F2 a) { return F2{fabsf(a.x), fabsf(a.y)}; }

// ---------------------------------------------------------------------------------------
// frame for a pair: symmetry reduction in (eq. (2)-(5)), sign restore out (eq. (8))
// ---------------------------------------------------------------------------------------
struct PairIn {
    F2 n1, n2, n3;   // sorted |n|, eq. (2)-(4)
    F2 n12;          // n1 + n2
    F2 hS;           // S/2
    F2 V2;           // 2 V = 2 min(V0, 1 - V0), saturated to [0, 1]
};

__device__ __forceinline__ PairIn pair_reduce(F2 V0, F2 nx, F2 ny, F2 nz) {
    PairIn in;
    const F2 a = abs2(nx), b = abs2(ny), c = abs2(nz);
    in.n1 = F2{min3(a.x, b.x, c.x), min3(a.y, b.y, c.y)};                       // eq. (2)
    in.n3 = F2{max3(a.x, b.x, c.x), max3(a.y, b.y, c.y)};                       // eq. (3)
    in.n2 = max2(min2(a, b), min2(max2(a, b), c));                              // eq. (4): median
    // eq. (5): V = 1/2 - |V0 - 1/2| = min(V0, 1 - V0); the saturation makes V0 < 0 act as 0
    // and V0 > 1 as 1
    const F2 V = min2(V0, fma2(V0, -1.0f, f2(1.0f)));
    in.V2 = F2{__saturatef(V.x + V.x), __saturatef(V.y + V.y)};
    in.n12 = add2(in.n1, in.n2);
    in.hS = mul2(add2(in.n12, in.n3), 0.5f);
    return in;
}

// d0 = sign(V0 - 1/2) (S/2 - d), eq. (8), from the residual r = S/2 - d >= 0: the sign is a bit
// operation, set when V0 <= 1/2.
__device__ __forceinline__ F2 pair_restore(F2 V0, F2 r) {
    const F2 t = fma2(V0, -1.0f, f2(0.5f));
    return F2{__uint_as_float(__float_as_uint(r.x) | (~__float_as_uint(t.x) & 0x80000000u)),
              __uint_as_float(__float_as_uint(r.y) | (~__float_as_uint(t.y) & 0x80000000u))};
}

// Last step of every method: the residual r = S/2 - d.  For cases (1)-(4) d <= S/2 is enforced
// (which also turns a NaN into r = 0); in case (5), d5 = V n3 + n12/2 (eq. (25)) gives
// r = S/2 - d5 = (n3 - W)/2 directly (W = 2 V n3 <= n3), one multiplication instead of forming d5.
// h = (n3 - W)/2 is passed in because the iterative methods use it as well.
__device__ __forceinline__ F2 pair_residual(const PairIn &in, F2 d, F2 W, F2 h) {
    return sel2(le2(in.n12, W), h, sub2(in.hS, min2(d, in.hS)));                // (5) | (1)-(4)
}

// A-priori (3)-vs-(4) decision on a pair: case (4) iff n3 < n12 and F3(e) > 0 (is_case4()).
// With z = n12 - W and e = n3 - n12, z + 2e = (n3 - W) + e, so
//   F3(e) = e^3 - 6 q e - 3 q z = e^3 - 3 q e - 3 q (n3 - W) = -3 [ q (n3 - W) + e (q - e^2/3) ],
// two FMAs on qn = q (n3 - W), which the case-(4) root needs anyway.
__device__ __forceinline__ B2 is_case4_2(F2 q, F2 e, F2 ee, F2 qn) {
    const F2 h = fma2(e, fma2(ee, -1.0f / 3.0f, q), qn);                         // -F3(e) / 3
    return B2{e.x < 0.0f && h.x < 0.0f, e.y < 0.0f && h.y < 0.0f};
}

template <int METHOD>
struct PairSolver;

// ---------------------------------------------------------------------------------------
// method 0, PLIC_FAST: analytic inverse (eq. (25)/(26)) for two cells at once.  Every closed
// form is evaluated and merged by select, (3)/(4) are chosen a priori and served by one
// trigonometric evaluation, and there is no branch at all, so the two cells of a pair (and
// the 32 lanes of a warp) share one instruction stream.  cbrt = ex2(lg2(x)/3).
// With R = 2 q (case 3) or u/4 (case 4) and rho = rsqrt(R), both cases read
//   d = base - 2 R rho g(C),   C = (3/4) rho {z | q (n3 - W) rho^2},   base = {n12 | S/2}
// [(3): 2 sqrt(2q) = 2 R rho, C3 = 3 z / (4 sqrt(2q));  (4): sqrt(u) = 2 R rho, C4 = 6 q (n3 - W) / u^(3/2)];
// the factor 2 is folded into g's Newton step.  Both roots are >= n2, which serves as the common
// floor (it also replaces a NaN from R = 0, i.e. n1 n2 flushed to zero, where the bracket
// [n2, n12] is narrower than fp32).
// ---------------------------------------------------------------------------------------
// The part of cases (3)/(4) that the analytic and the SZ kernel share: R, rho, the argument C of
// the trigonometric root, the case flag and h = (n3 - W)/2.
struct Trig34 {
    F2 R, rho, C, h;
    B2 c4;
};
__device__ __forceinline__ Trig34 trig34(const PairIn &in, F2 W) {
    Trig34 t;
    const F2 q = mul2(in.n1, in.n2);
    const F2 e = sub2(in.n3, in.n12);
    const F2 z = sub2(in.n12, W);
    const F2 ee = mul2(e, e);
    const F2 n3mW = sub2(in.n3, W);
    const F2 qn = mul2(q, n3mW);
    t.h = mul2(n3mW, 0.5f);
    t.c4 = is_case4_2(q, e, ee, qn);
    t.R = sel2(t.c4, fma2(ee, -0.25f, q), add2(q, q));                          // u/4 | 2 q
    t.rho = rsqrt2(t.R);
    const F2 K4 = mul2(qn, mul2(t.rho, t.rho));
    t.C = mul2(sel2(t.c4, K4, z), mul2(t.rho, 0.75f));
    return t;
}

template <>
struct PairSolver<ANALYTIC> {
    static __device__ __forceinline__ F2 residual(const PairIn &in) {
        const F2 n1 = in.n1, n2 = in.n2, n12 = in.n12;
        const F2 W = mul2(in.V2, in.n3);                                        // 2 V n3
        const F2 Wn2 = mul2(W, n2);                                             // x / 3, x = 6 V n2 n3
        const F2 s1 = mul2(n1, n1);
        const F2 t1 = fma2(s1, -1.0f / 3.0f, Wn2);                              // (x - n1^2) / 3
        // (2) and (1): d1 = cbrt(x n1) = 2^(lg2(Wn2 n1)/3 + lg2(3)/3).  The radicand of d2 needs no
        // clamp: where (2) is selected, t1 >= 0, and Wn2 - n1^2/12 >= Wn2 - n1^2/3 = t1 holds for
        // the rounded FMAs too (monotone in the addend); elsewhere its NaN is dropped by the select
        const F2 d2 = fma2(n1, 0.5f, sqrt2(fma2(s1, -1.0f / 12.0f, Wn2)));
        const F2 d1 = ex2_2(fma2(lg2_2(mul2(Wn2, n1)), 1.0f / 3.0f, f2(0.528320834f)));
        F2 d = sel2(lt2(t1, f2(0.0f)), d1, d2);                                 // x < n1^2
        // (3)/(4)
        const Trig34 t = trig34(in, W);
        const F2 ng2 = neg_sin_third_asin_fast2<true>(t.C);                     // -2 g(C)
        const F2 d34 = max2(fma2(mul2(t.R, t.rho), ng2, sel2(t.c4, in.hS, n12)), n2);   // floor; drops NaN
        d = sel2(gt2(t1, mul2(n2, sub2(n2, n1))), d34, d);                      // x > n1^2 + 3 n2 (n2 - n1)
        return pair_residual(in, d, W, t.h);
    }
};

// ---------------------------------------------------------------------------------------
// method 1, PLIC_FAST: Scardovelli-Zaleski (sect. 2.4) on a pair, branch-free: thresholds
// multiplied through, (5) and (2) tested first, root
//   alpha = 2 sqrt(p0) cos(acos(q0 / p0^(3/2)) / 3 + 4 pi / 3) - a2/3
// with the collapsed p0, q0 of Precise<SZ> (plic_methods.cuh).  Micro-optimised further:
//   * the L1 normalisation m_i = n_i / S is folded away: every quantity of the method is homogeneous
//     in n (alpha S = d, 4 p0 S^2 = R', q0 / p0^(3/2) is scale free), so the kernel works on the n_i
//     and never divides by S -- the precise kernel (Precise<SZ>) keeps the normalisation literally;
//   * with R = p0 S^2 (= 2 q in case (3), u/4 in case (4)) and rho = rsqrt(R):
//     2 sqrt(p0) S = 2 R rho and q0 / p0^(3/2) = (3/4) rho {z | q (n3 - W) rho^2}  (trig34());
//   * the (3)-vs-(4) threshold w6 >= 6 m1 m2 m3 v3 is the sign of the case-(3)
//     cubic at alpha = m3, a polynomial in m12 - m3 (is_case4_2), instead of the v3 polynomial;
//   * the tests (1)/(2)/(3,4) in the scaled variable t1 = W n2 - n1^2 / 3;
//   * acos by sqrt(1-x) Q5(x), the angle's 1/3 and the 4 pi / 3 in one FMA, cos on the SFU.
// What distinguishes it from the analytic kernel is acos + cos in place of the sin(asin(.)/3)
// polynomial.
// ---------------------------------------------------------------------------------------
// acos(x) for x in [0, 0.9] as sqrt(1-x) * Q5(x), |err| < 1.2e-6 (minimax fit on [0, 1],
// fit_coefficients.py).  No clamps: for a cell of case (3)/(4) the argument is <= 0.884 (DESIGN.md,
// "trig range"); elsewhere a NaN is dropped by the floor of the root.
__device__ __forceinline__ F2 acos_fast2(F2 x) {
    F2 p = fma2(x, f2(-0.004337173733f), f2(0.01934827404f));
    p = fma2(p, x, f2(-0.04495724702f));
    p = fma2(p, x, f2(0.08787565452f));
    p = fma2(p, x, f2(-0.2145122723f));
    p = fma2(p, x, f2(1.570795206f));
    return mul2(sqrt2(fma2(x, -1.0f, f2(1.0f))), p);
}

template <>
struct PairSolver<SZ> {
    static __device__ __forceinline__ F2 residual(const PairIn &in) {
        const F2 n1 = in.n1, n2 = in.n2, n12 = in.n12;
        const F2 W = mul2(in.V2, in.n3);                                        // 2 w m3 S
        const F2 Wn2 = mul2(W, n2);                                             // x S^2 / 3, x = 6 w m2 m3
        const F2 s1 = mul2(n1, n1);
        const F2 t1 = fma2(s1, -1.0f / 3.0f, Wn2);                              // (x - m1^2) S^2 / 3
        // (2): v1 <= w <= v2, and (1): w < v1  <=>  x < m1^2;  alpha S = cbrt(w6 S^3), w6 S^3 = 3 Wn2 n1
        const F2 d2 = fma2(n1, 0.5f, sqrt2(fma2(s1, -1.0f / 12.0f, Wn2)));
        const F2 d1 = ex2_2(fma2(lg2_2(mul2(Wn2, n1)), 1.0f / 3.0f, f2(0.528320834f)));
        F2 d = sel2(lt2(t1, f2(0.0f)), d1, d2);
        // (3)/(4)
        const Trig34 t = trig34(in, W);                                         // C = q0 / p0^(3/2)
        // cos(theta + 4 pi/3) evaluated as cos(theta - 2 pi/3): same angle, |arg| < pi
        const F2 co = cos2(fma2(acos_fast2(t.C), 1.0f / 3.0f, f2(-2.0943951f)));
        const F2 d34 = max2(fma2(mul2(t.R, add2(t.rho, t.rho)), co, sel2(t.c4, in.hS, n12)), n2);   // floor; drops NaN
        d = sel2(gt2(t1, mul2(n2, sub2(n2, n1))), d34, d);
        return pair_residual(in, d, W, t.h);
    }
};

// ---------------------------------------------------------------------------------------
// method 2, PLIC_FAST: Newton-Raphson (sect. 2.5) on a pair.  One unrolled loop on
// F(tau) = tau^3 - p tau - r serves (1), (3) and (4) with selected coefficients; every lane runs
// it (no branch), (2) and (5) are closed forms, division by SFU reciprocal.
//   * The iteration runs on sigma = -tau >= 0 with F / 2:
//       sigma <- (sigma^3 + rn) / (3/2 sigma^2 + nh),   nh = -p/2,  rn = -r/2,
//     one instruction less than the textbook step (no 2 tau^2); the negated form makes rn a single
//     product: rn = (-3/2 q) {z | (n3 - W)/2}.
//   * Start: the Newton step from tau = 0 in closed form, sigma_0 = r/p = rn / nh.  tau = 0 lies
//     right of the root in the region where F is decreasing and concave (F(0) = -r <= 0,
//     F' = 3 tau^2 - p < 0 on [root, 0]), so the iteration is monotone from there; 3 more steps
//     leave 6e-8 (the round-1 kernel started at the top of the bracket and needed 4 for 4e-8).
//   * Case (1), d^3 = 6 V n1 n2 n3 = 3 Wn2 n1: nh = 0, rn = -3/2 Wn2 n1, sigma_0 = -seed with the
//     integer-arithmetic cube-root seed (exponent / 3), d = -sigma; 3 steps from a seed within 4 %
//     are exact to rounding.
// ---------------------------------------------------------------------------------------
// start value for -cbrt(3 k3), k3 > 0: cbrt_seed() with the factor 3 folded into the constant
// (+ lg2(3)/3 in the exponent field; 0x2a952e80 minimises the maximum relative error over
// [1e-30, 1]: 3.9 %) and the sign bit set
__device__ __forceinline__ float neg_cbrt3_seed(float k3) {
    // k3 >= 0: unsigned high multiply = bits / 3 (one IMAD.HI, no sign fix-up)
    return __uint_as_float((__umulhi(__float_as_uint(k3), 0x55555556u) + 0x2a952e80u) | 0x80000000u);
}

template <>
struct PairSolver<NEWTON> {
    static __device__ __forceinline__ F2 residual(const PairIn &in) {
        const F2 n1 = in.n1, n2 = in.n2, n3 = in.n3, n12 = in.n12;
        const F2 W = mul2(in.V2, n3);
        const F2 Wn2 = mul2(W, n2);
        const F2 s1 = mul2(n1, n1);
        const F2 t1 = fma2(s1, -1.0f / 3.0f, Wn2);                              // (x - n1^2) / 3
        const B2 c1 = lt2(t1, f2(0.0f));                                        // x < n1^2
        const B2 c34 = gt2(t1, mul2(n2, sub2(n2, n1)));                         // x > n1^2 + 3 n2 (n2 - n1)
        const F2 d2 = fma2(n1, 0.5f, sqrt2(fma2(s1, -1.0f / 12.0f, Wn2)));
        const F2 q = mul2(n1, n2);
        const F2 e = sub2(n3, n12);
        const F2 z = sub2(n12, W);
        const F2 ee = mul2(e, e);
        const F2 n3mW = sub2(n3, W);
        const F2 h = mul2(n3mW, 0.5f);                                          // (n3 - W)/2
        const B2 c4 = is_case4_2(q, e, ee, mul2(q, n3mW));
        const F2 zero = f2(0.0f);
        const F2 qm = mul2(q, -1.5f);
        const F2 nh34 = sel2(c4, fma2(ee, 0.375f, qm), add2(qm, qm));           // -3u/8 | -3q
        const F2 rn34 = mul2(qm, sel2(c4, h, z));                               // -3/4 q (n3 - W) | -3/2 q z
        const F2 k3 = mul2(Wn2, n1);                                            // 2 V n1 n2 n3
        const F2 nh = sel2(c1, zero, nh34);
        const F2 rn = sel2(c1, mul2(k3, -1.5f), rn34);
        F2 sig = sel2(c1, F2{neg_cbrt3_seed(k3.x), neg_cbrt3_seed(k3.y)}, mul2(rn34, rcp2(nh34)));
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            const F2 s2 = mul2(sig, sig);
            sig = mul2(fma2(s2, sig, rn), rcp2(fma2(s2, 1.5f, nh)));
        }
        const F2 d34 = max2(fma2(sig, -1.0f, sel2(c4, in.hS, n12)), n2);        // floor; drops NaN
        F2 d = sel2(c34, d34, d2);
        d = sel2(c1, F2{-sig.x, -sig.y}, d);
        return pair_residual(in, d, W, h);
    }
};

// ---------------------------------------------------------------------------------------
// method 3, PLIC_FAST: nested intervals (sect. 2.5) on a pair: kNestedFastHalvings = 16 fixed
// halvings of the bracket [lo, hi] of the depressed cubic F for (3)/(4); closed forms for (1),
// (2), (5).  F is decreasing on the bracket, F(lo) >= 0 >= F(hi).
// Accuracy is bought per halving: after N halvings the centre is within w 2^-(N+1) of the root,
// w = hi - lo <= n1 <= 0.577, i.e. |err| <= 4.4e-6 for N = 16 -- 4.5 times inside the 2e-5 bar, and
// the forward-volume residual (dV/dd0 = area of the cut <= sqrt 2) <= 6.3e-6.  Rounds 1-2 ran
// N = 20 (|err| <= 2.9e-7 observed) at 20 x 8 issue slots per pair, which left the kernel at half
// its HBM roofline; the precise kernel (no PLIC_FAST) still halves until the fp32 midpoint stops
// moving, as the paper's listing does.  -DPLIC_NESTED_FAST_HALVINGS=20
// rebuilds the old trade.
//
// The halving runs in the scaled variable y = tau / (hi - lo), in which the bracket has unit
// width, and carries the interval's CENTRE c instead of its lower end:
//     G(y) = y^3 - P y - R,   P = p / w^2,  R = r / w^3,  w = hi - lo      (G = F / w^3)
//     c_0 = lo/w + 1/2,   c_{k+1} = c_k + copysign(2^-(k+2), G(c_k))
// G(c) > 0 means the root lies right of c.  The interval after k steps is c_k +- 2^-(k+1), the
// same sequence of intervals as (lo, hi) bisection.  The step sizes are compile-time
// constants, so one halving costs two packed FMAs, one sign transfer per half (LOP3:
// (G & 0x80000000) | 2^-(k+2)) and one packed add -- 5 issued instructions per pair instead of
// the 8 of the compare-and-select form (FMUL2, FADD2, 2 FFMA2, 2 FSETP, 2 FSEL).  Rounding: c
// may be large when the bracket is narrow and far from 0 (|lo| >> w), but ulp(c) w = ulp(lo),
// the resolution tau has anyway.  w = 0 or a flushed product gives NaN or 0, which the floor
// n2 replaces (the bracket is then narrower than fp32).
// ---------------------------------------------------------------------------------------
// The sign mask is read from constant memory so that it sits in a register and the LOP3's one
// immediate slot is free for the step size (as a literal mask, ptxas moves every step constant
// into a register first: one more instruction per step).
__constant__ unsigned kSignMask = 0x80000000u;
__device__ __forceinline__ unsigned sign_mask_register() {
    unsigned m;
    asm volatile("{ .reg .u64 a; cvta.to.const.u64 a, %1; ld.const.u32 %0, [a]; }" : "=r"(m) : "l"(&kSignMask));
    return m;
}

template <unsigned STEP_BITS>
__device__ __forceinline__ float signed_step(float G, unsigned mask) {
    unsigned r;
    asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=r"(r) : "r"(__float_as_uint(G)), "r"(mask), "n"(STEP_BITS));
    return __uint_as_float(r);
}

#ifndef PLIC_NESTED_FAST_HALVINGS
#define PLIC_NESTED_FAST_HALVINGS 16
#endif
constexpr int kNestedFastHalvings = PLIC_NESTED_FAST_HALVINGS;
static_assert(kNestedFastHalvings >= 14 && kNestedFastHalvings <= 22,
              "14 halvings are 1.8e-5 (no margin to the 2e-5 bar), beyond 22 the step falls below an fp32 ulp of c");

template <int K, int N>
struct NestedSteps {
    static __device__ __forceinline__ void run(F2 &c, const F2 &nP, const F2 &nR, unsigned mask) {
        const F2 G = fma2(fma2(c, c, nP), c, nR);
        constexpr unsigned step = (unsigned)(127 - (K + 2)) << 23;              // bits of 2^-(K+2)
        c = add2(c, F2{signed_step<step>(G.x, mask), signed_step<step>(G.y, mask)});
        NestedSteps<K + 1, N>::run(c, nP, nR, mask);
    }
};
template <int N>
struct NestedSteps<N, N> {
    static __device__ __forceinline__ void run(F2 &, const F2 &, const F2 &, unsigned) {}
};

template <>
struct PairSolver<NESTED> {
    static __device__ __forceinline__ F2 residual(const PairIn &in) {
        const F2 n1 = in.n1, n2 = in.n2, n3 = in.n3, n12 = in.n12;
        const F2 W = mul2(in.V2, n3);
        const F2 Wn2 = mul2(W, n2);                                             // x / 3
        const F2 s1 = mul2(n1, n1);
        const F2 t1 = fma2(s1, -1.0f / 3.0f, Wn2);                              // (x - n1^2) / 3
        const F2 d2 = fma2(n1, 0.5f, sqrt2(fma2(s1, -1.0f / 12.0f, Wn2)));
        const F2 d1 = ex2_2(fma2(lg2_2(mul2(Wn2, n1)), 1.0f / 3.0f, f2(0.528320834f)));
        F2 d = sel2(lt2(t1, f2(0.0f)), d1, d2);
        const F2 q = mul2(n1, n2);
        const F2 e = sub2(n3, n12);
        const F2 z = sub2(n12, W);
        const F2 ee = mul2(e, e);
        const F2 n3mW = sub2(n3, W);
        const F2 h = mul2(n3mW, 0.5f);                                          // (n3 - W)/2
        const B2 c4 = is_case4_2(q, e, ee, mul2(q, n3mW));
        const F2 zero = f2(0.0f);
        const F2 qm = mul2(q, -3.0f);
        const F2 np = sel2(c4, fma2(ee, 0.75f, qm), add2(qm, qm));              // -p: -3u/4 | -6q
        const F2 nr = mul2(qm, sel2(c4, h, z));                                 // -r: -3/2 q (n3 - W) | -3 q z
        const F2 lo = sel2(c4, sub2(n3, in.hS), mul2(n1, -1.0f));
        const F2 hi = sel2(c4, zero, min2(e, zero));
        const F2 w = sub2(hi, lo);
        const F2 iw = rcp2(w);
        const F2 iw2 = mul2(iw, iw);
        const F2 nP = mul2(np, iw2);                                            // -p / w^2
        const F2 nR = mul2(mul2(nr, iw), iw2);                                  // -r / w^3
        F2 c = fma2(lo, iw, f2(0.5f));
        NestedSteps<0, kNestedFastHalvings>::run(c, nP, nR, sign_mask_register());
        const F2 d34 = max2(fma2(c, w, sel2(c4, in.hS, n12)), n2);              // floor; drops NaN
        d = sel2(gt2(t1, mul2(n2, sub2(n2, n1))), d34, d);
        return pair_residual(in, d, W, h);
    }
};

// One pair through frame and method: eq. (2)-(5) -> method -> eq. (8).
template <int METHOD>
__device__ __forceinline__ F2 solve_pair_fast(F2 V0, F2 nx, F2 ny, F2 nz) {
    const PairIn in = pair_reduce(V0, nx, ny, nz);
    return pair_restore(V0, PairSolver<METHOD>::residual(in));
}

// ---------------------------------------------------------------------------------------
// forward map V0(d0, n) for two cells at once: eq. (2)-(4), (7), (11), (6)   (Listing 1,
// PAPER.md:71-92), branch-free.  Case (5) is tested first and case (2) is in its n1-free form,
// so n1 = 0 and n1 = n2 = 0 never divide by zero (caption of Listing 1).  Cases (3) and (4) are
// evaluated in forms expanded around d = n12 resp. d = S/2,
//   (3): V = (n12/2 + t - t^3/(6 q)) / n3,          t = d - n12 in [-n1, 0]
//   (4): V = 1/2 + s (3 u/4 - s^2) / (3 q n3),      s = d - S/2 in [-n1/2, 0],  u = 4 q - (n3 - n12)^2
// instead of the fdim-merged difference of cubes of Listing 1: that difference cancels to
// ~eps d^3/(6 n1 n2 n3) in fp32, i.e. 4e-3 for n1 = 1e-6 ("forward map").
// All five cases are brought to one quotient
//   V = top + num / den,   top = 1/2 for (4), (5) and 0 for (1)-(3):
//   (1) d^3                                   / (6 q n3)
//   (2) 3 d (d - n1) + n1^2                   / (6 n2 n3)
//   (3) 6 q (n12/2 + t) - t^3                 / (6 q n3)
//   (4) s (3/2 u - 2 s^2)                     / (6 q n3)
//   (5) -|d0|                                 / n3               [(d - n12/2)/n3 = 1/2 - |d0|/n3]
// so one division serves every case.  It is a reciprocal (SFU) with one Newton correction of
// the quotient, i.e. within 1-2 ulp of the IEEE quotient.  den is floored at 1e-37: a zero
// normal then gives 1/2 - |d0| / 1e-37 -> 1/2 for d0 = 0 and 0 otherwise, as documented.
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ F2 volume_pair(F2 d0, F2 nx, F2 ny, F2 nz) {
    const F2 a = abs2(nx), b = abs2(ny), c = abs2(nz);
    const F2 n1 = F2{min3(a.x, b.x, c.x), min3(a.y, b.y, c.y)};
    const F2 n3 = F2{max3(a.x, b.x, c.x), max3(a.y, b.y, c.y)};
    const F2 n2 = max2(min2(a, b), min2(max2(a, b), c));
    const F2 n12 = add2(n1, n2);
    const F2 hS = mul2(add2(n12, n3), 0.5f);
    const F2 ad0 = abs2(d0);
    const F2 d = F2{fmaxf(hS.x - ad0.x, 0.0f), fmaxf(hS.y - ad0.y, 0.0f)};        // eq. (7)
    const F2 q = mul2(n1, n2);
    const F2 q6 = mul2(q, 6.0f);
    // (1), (2)
    const F2 num1 = mul2(mul2(d, d), d);
    const F2 num2 = fma2(mul2(d, 3.0f), sub2(d, n1), mul2(n1, n1));
    // (3): 6 q (n12/2 + t) - t^3 with nt = -t = n12 - d in [0, n1]
    const F2 nt = sub2(n12, d);
    const F2 num3 = fma2(fma2(n12, 0.5f, mul2(nt, -1.0f)), q6, mul2(mul2(nt, nt), nt));
    // (4): s (3/2 u - 2 s^2), 3/2 u = 6 q - 3/2 e^2
    const F2 s_ = sub2(d, hS);
    const F2 e = sub2(n3, n12);
    const F2 u15 = fma2(mul2(e, e), -1.5f, q6);
    const F2 num4 = mul2(s_, fma2(mul2(s_, s_), -2.0f, u15));
    // case selection: (5) first, then (1), (2), (3), else (4)
    const B2 c5 = B2{d.x >= n12.x, d.y >= n12.y};
    const B2 c1 = lt2(d, n1);
    const B2 c2 = le2(d, n2);
    const B2 c3 = le2(d, n3);
    F2 num = sel2(c3, num3, num4);
    num = sel2(c2, num2, num);
    num = sel2(c1, num1, num);
    num = sel2(c5, F2{-ad0.x, -ad0.y}, num);
    const B2 use_n2 = andnot2(c2, c1);                                           // case (2)
    F2 den = mul2(mul2(n3, 6.0f), sel2(use_n2, n2, q));
    den = max2(sel2(c5, n3, den), 1e-37f);
    const B2 top = B2{c5.x || !c3.x, c5.y || !c3.y};                             // (4) or (5)
    // V = top + num/den:  nr = -1/den,  nv = -num/den,  corrected by err = num - den (num/den)
    const F2 nr = F2{mufu_rcp(-den.x), mufu_rcp(-den.y)};
    const F2 nv = mul2(num, nr);
    const F2 nv2 = fma2(fma2(den, nv, num), nr, nv);
    F2 V = fma2(nv2, -1.0f, sel2(top, f2(0.5f), f2(0.0f)));
    V = min2(max2(V, 0.0f), f2(0.5f));
    const F2 Vc = fma2(V, -1.0f, f2(1.0f));
    return sel2(gt2(d0, f2(0.0f)), Vc, V);                                       // eq. (6)
}

// ---------------------------------------------------------------------------------------
// plane-sphere intersection (sect. 3): unit-volume sphere, r = (3/(4 pi))^(1/3)
// (eq. (34)).  Forward eq. (37) in cap form: with a = r - |d0| the smaller cap has volume
// pi/3 a^2 (3r - a), mirrored for d0 > 0 -- the same polynomial as eq. (37), evaluated from the
// near pole so that both ends keep full relative accuracy.
// Inverse eq. (38): atan2(2 sqrt(V0 - V0^2), 2 V0 - 1) = acos(2 V0 - 1) because the two arguments
// lie on the unit circle.  With V = min(V0, 1 - V0) and psi = asin(sqrt V)/3 in [0, pi/12]
// (acos(1 - 2V) = 2 asin(sqrt V)) the cap height is
//   a = r - |d0| = 2r (sin(pi/6) - sin(pi/6 - 2 psi)) = 4r sin(psi) cos(pi/6 - psi),
// which has no cancellation at V -> 0 (eq. (38) as printed loses the digits of V0 in 2 V0 - 1).
// sin(psi) = g(sqrt V) is the same sin(asin(C)/3) as in cases (3)/(4) of the cube, C <= 0.7072.
// ---------------------------------------------------------------------------------------
constexpr float kSphereR = 0.62035048f;                 // fp32((3/(4 pi))^(1/3)), eq. (34)
constexpr float kSphereRlo = 1.08197492e-8f;            // r - kSphereR: keeps small caps accurate

__device__ __forceinline__ F2 sphere_volume_pair(F2 d0) {
    const F2 ad = abs2(d0);
    // a = r - |d0|: the difference with fp32(r) is exact near the pole, the tail of r is added after
    const F2 a = F2{fmaxf((kSphereR - ad.x) + kSphereRlo, 0.0f), fmaxf((kSphereR - ad.y) + kSphereRlo, 0.0f)};
    // pi/3 a^2 (3r - a)
    const F2 V = mul2(mul2(a, a), fma2(a, -1.04719755f, f2(3.0f * kSphereR * 1.04719755f)));
    return sel2(gt2(d0, f2(0.0f)), fma2(V, -1.0f, f2(1.0f)), V);
}

__device__ __forceinline__ F2 sphere_solve_pair_fast(F2 V0) {
    const F2 V = sat2(min2(V0, fma2(V0, -1.0f, f2(1.0f))));
    const F2 nsin = neg_sin_third_asin_fast2<false>(sqrt2(V));                          // -sin(psi)
    const F2 cosp = sqrt2(fma2(mul2(nsin, -1.0f), nsin, f2(1.0f)));              // cos(psi)
    // a = 4r sin(psi) (sqrt(3)/2 cos(psi) + 1/2 sin(psi))
    const F2 a = mul2(mul2(nsin, -4.0f * kSphereR), fma2(cosp, 0.866025404f, mul2(nsin, -0.5f)));
    const F2 r = F2{fmaxf(kSphereR - a.x, 0.0f), fmaxf(kSphereR - a.y, 0.0f)};
    const F2 t = fma2(V0, -1.0f, f2(0.5f));
    return F2{__uint_as_float(__float_as_uint(r.x) | (~__float_as_uint(t.x) & 0x80000000u)),
              __uint_as_float(__float_as_uint(r.y) | (~__float_as_uint(t.y) & 0x80000000u))};
}

// precise: IEEE sqrt, libm asin/sin/cos
__device__ __forceinline__ float sphere_solve_cell(float V0) {
    const float V = fmaxf(fminf(V0, 1.0f - V0), 0.0f);
    const float psi = asinf(fminf(sqrtf(V), 1.0f)) * (1.0f / 3.0f);
    const float a = 4.0f * kSphereR * sinf(psi) * cosf(0.523598776f - psi);
    const float r = fmaxf(kSphereR - a, 0.0f);
    return V0 > 0.5f ? r : -r;
}

}  // namespace plic
