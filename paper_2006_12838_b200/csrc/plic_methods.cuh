// plic_methods.cuh -- per-cell fp32 device functions of the PLIC hot path (sm_100a).
//
// PAPER.md = /root/reference/PAPER.md (arxiv 2006.12838).  Notation follows the paper:
//   n1 <= n2 <= n3   mirrored, sorted normal components        eq. (2)-(4)
//   V in [0, 1/2]    reduced volume                            eq. (5),
//   d in [0, S/2]    reduced offset from the cube corner       eq. (7),
//   (1)..(5)         the five intersection cases               eq. (11),
// and, as shorthands used throughout:
//   n12 = n1+n2, S = n1+n2+n3, q = n1 n2, W = 2 V n3, z = n12 - W, e = n3 - n12,
//   x = 6 V n2 n3 = 3 W n2,  u = 4 q - e^2  ( = S^2 - 2 sum n_i^2; = t4/9 of eq. (19) when |n|=1 ).
//
// This file holds the precise (FAST = false) kernels: IEEE division and square root, CUDA
// libm cbrt/asin/acos/sin/cos, branches in the paper's order.  The PLIC_FAST kernels are in
// plic_packed.cuh (two cells per instruction, branch-free, SFU roots); cbrt_seed() here
// serves both.  Each method is `Solver<METHOD, false>::reduced_offset(n1, n2, n3, V) -> d`; the
// frame solve_cell() does the symmetry reduction before and the sign restore (eq. (8)) after.  The bodies of
// the paper's Listings 1, 2, 4, 5, 6 are not in PAPER.md (captions only) and Listing 3 is
// truncated, so every method is built from the equations; DESIGN.md lists the readings.
//
// Cases (3) and (4) are cubics in d.  All methods use them in depressed form
//   F(tau) = tau^3 - p tau - r = 0,  d = base + tau:
//   case (3): base = n12, p = 6 q,     r = 3 q z,          tau in [-n1, min(0, e)]
//   case (4): base = S/2, p = 3 u / 4, r = 3 q (n3 - W)/2, tau in [n3 - S/2, 0]
// (expand eq. (11) around d = n12 resp. d = S/2), because every coefficient is then a
// product of small quantities and no cancellation of O(1) terms occurs when n1 is small.
// The trigonometric root of these cubics is
//   tau = -2 sqrt(p/3) sin(asin(C)/3),  C = (r/2) (3/p)^(3/2),
// which is eq. (12) with atan2(y,x) = acos(C) and pi/6 - acos(C)/3 = asin(C)/3:
//   case (3): d = n12 - 2 sqrt(2 q) sin(asin(C3)/3), C3 = 3 z / (4 sqrt(2 q))
//   case (4): d = S/2 - sqrt(u)     sin(asin(C4)/3), C4 = 6 q (n3 - W) / u^(3/2).
// Which of (3)/(4) applies is decided a priori by the sign of F3(e) (d3 <= n3  <=>  F3(e) <= 0,
// F3 being decreasing on [-n1, 0]), or a posteriori by d3 <= n3 as the paper does
// (PAPER.md:151), where noted.
#pragma once
#include "plic_math.cuh"

namespace plic {

enum : int { ANALYTIC = 0, SZ = 1, NEWTON = 2, NESTED = 3, KAWANO = 4 };

// ---------------------------------------------------------------------------------------
// shared pieces
// ---------------------------------------------------------------------------------------

// A-priori (3)-vs-(4) decision: case (4) iff n3 < n12 and F3(e) > 0.
__device__ __forceinline__ bool is_case4(float q, float e, float ee, float z) {
    const float h = fmaf(fmaf(-6.0f, q, ee), e, -3.0f * (q * z));
    return (e < 0.0f) && (h > 0.0f);
}

// Newton-Raphson on F(tau) = tau^3 - p tau - r:  tau <- (2 tau^3 + r) / (3 tau^2 - p).
template <bool FAST, int ITERS>
__device__ __forceinline__ float newton_cubic(float p, float r, float tau) {
#pragma unroll
    for (int i = 0; i < ITERS; ++i) {
        const float t2 = tau * tau;
        tau = Math<FAST>::div(fmaf(2.0f * t2, tau, r), fmaf(3.0f, t2, -p));
    }
    return tau;
}

// Start value for the cube root of k > 0: exponent/3 by integer arithmetic (relative error
// <= 3.2 %; the constant minimises the maximum error over [1e-30, 1]).
__device__ __forceinline__ float cbrt_seed(float k) {
    return __int_as_float(__float_as_int(k) / 3 + 0x2a510680);
}

// ---------------------------------------------------------------------------------------
// The precise methods in three pieces.  A random warp holds all five intersection cases
// ("GPUs are especially bad at branching"), so each method is split into
//   cheap()    cases (5) and (2): two closed forms, evaluated for every cell without a branch,
//              and the case decision `kind` (a priori, eq. (26) with the misprint corrected);
//   heavy_a()  cases (3)/(4): the expensive root (trigonometric, Newton-Raphson, bisection),
//              one code path for both cases with (3)/(4) chosen a priori by is_case4();
//   heavy_b()  case (1): the cube root (libm cbrtf, or Newton-Raphson on d^3 = 6 V n1 n2 n3).
// The scalar form reduced_offset() branches on `kind` in the paper's order (5)->(2)->(1)->(3)->(4);
// the streaming body (map_compact in plic_kernels.cu) runs cheap() for all cells, collects the
// heavy cells of a 1024-cell tile in shared memory and evaluates them in dense warps.  Both
// call the same three functions, whose results are formed by fmaf / min / max / select or
// round-to-nearest intrinsics only, so that no multiply is contracted with an add of the caller
// and the two forms agree bitwise.
// ---------------------------------------------------------------------------------------
// `kind` doubles as the increment of map_compact's packed queue counter (heavy-A entries in the
// low half, heavy-B entries in the high half)
enum : int { KIND_DONE = 0, KIND_HEAVY_A = 1, KIND_HEAVY_B = 0x10000 };

template <int METHOD>
struct Precise;

// Cases (5), (2) and the case decision in n-space (analytic, Newton-Raphson, nested intervals).
struct CheapN {
    static __device__ __forceinline__ float cheap(float n1, float n2, float n3, float V, int &kind) {
        const float n12 = n1 + n2;
        const float W = 2.0f * V * n3;
        const float x = 3.0f * W * n2;                                     // 6 V n2 n3
        const float s1 = n1 * n1;
        const bool c5 = n12 <= W;                                          // (5) eq. (26)
        const bool c1 = x < s1;                                            // (1)
        // (2): n1^2 <= 6 V n2 n3 <= n1^2 + 3 n2 (n2 - n1)   [eq. (26), misprint corrected]
        const bool c2 = x <= fmaf(3.0f * n2, n2 - n1, s1);
        const float d5 = fmaf(V, n3, 0.5f * n12);
        const float d2 = fmaf(0.5f, n1, sqrtf(fmaxf(fmaf(W, n2, -s1 * (1.0f / 12.0f)), 0.0f)));
        kind = c5 ? KIND_DONE : (c1 ? KIND_HEAVY_B : (c2 ? KIND_DONE : KIND_HEAVY_A));
        return c5 ? d5 : d2;
    }
    static __device__ __forceinline__ float k6(float n1, float n2, float n3, float V) {
        return __fmul_rn(3.0f * (2.0f * V * n3) * n2, n1);                 // 6 V n1 n2 n3
    }
};

// depressed cubic of case (3) or (4), chosen a priori: F(tau) = tau^3 - p tau - r on [lo, hi],
// d = base + tau, d >= floor
struct Cubic34 {
    float p, r, lo, hi, base, floor;
};
__device__ __forceinline__ Cubic34 cubic34(float n1, float n2, float n3, float V) {
    const float n12 = n1 + n2;
    const float W = 2.0f * V * n3;
    const float q = n1 * n2;
    const float e = n3 - n12;
    const float z = n12 - W;
    const float ee = e * e;
    const bool c4 = is_case4(q, e, ee, z);
    const float hS = 0.5f * (n12 + n3);
    Cubic34 c;
    c.p = c4 ? 0.75f * fmaf(4.0f, q, -ee) : 6.0f * q;
    c.r = c4 ? 1.5f * q * (n3 - W) : 3.0f * q * z;
    c.lo = c4 ? n3 - hS : -n1;
    c.hi = c4 ? 0.0f : fminf(e, 0.0f);
    c.base = c4 ? hS : n12;
    c.floor = c4 ? n3 : n2;
    return c;
}

// ---------------------------------------------------------------------------------------
// method 0: the paper's analytic inverse, eq. (25)/(26)
//   (3): d = n12 - 2 sqrt(2 q) g(C3), C3 = 3 z / (4 sqrt(2 q))
//   (4): d = S/2 - sqrt(u)     g(C4), C4 = 6 q (n3 - W) / u^(3/2),   g(C) = sin(asin(C)/3)
// as one evaluation with A = 2 q or u: IEEE sqrt and division, libm asinf / sinf.  The paper
// decides (3)-vs-(4) a posteriori by d3 <= n3, which costs case-(4) cells a
// second trigonometric root; the a-priori test is equivalent (d3 <= n3 <=> F3(e) <= 0).
// ---------------------------------------------------------------------------------------
template <>
struct Precise<ANALYTIC> : CheapN {
    static __device__ __forceinline__ float heavy_a(float n1, float n2, float n3, float V) {
        typedef Math<false> M;
        const float n12 = n1 + n2;
        const float W = 2.0f * V * n3;
        const float q = n1 * n2;
        const float e = n3 - n12;
        const float z = n12 - W;
        const float ee = e * e;
        const bool c4 = is_case4(q, e, ee, z);
        const float A = c4 ? fmaf(4.0f, q, -ee) : q + q;                   // u or 2 q
        const float sA = M::sqrt(A);
        const float num = c4 ? 6.0f * q * (n3 - W) : 0.75f * z;
        const float C = M::div(num, c4 ? A * sA : sA);
        const float amp = c4 ? -sA : -2.0f * sA;
        const float d = fmaf(amp, M::sin_third_asin(C), c4 ? 0.5f * (n12 + n3) : n12);
        return fmaxf(d, c4 ? n3 : n2);                                     // bracket floor; drops NaN
    }
    static __device__ __forceinline__ float heavy_b(float n1, float n2, float n3, float V) {
        return Math<false>::cbrt(k6(n1, n2, n3, V));                       // (1)
    }
};

// ---------------------------------------------------------------------------------------
// method 1: Scardovelli-Zaleski, edge-case complete and micro-optimised (sect. 2.4)
//
// L1-normalised m_i = n_i / S, alpha = d / S, w = V.  Cases chosen a priori
// from volume thresholds multiplied through so that nothing divides by m1 or m2, with (5)
// and (2) tested first.  The cubic of Listing 3,
//   case (3): a2 = -3 m12, a1 = 3 (m1^2+m2^2),    a0 = w6 - m1^3 - m2^3
//   case (4): a2 = -3/2,   a1 = 3/2 sum m_i^2,    a0 = (w6 - sum m_i^3)/2,   w6 = 6 m1 m2 m3 w
// is solved by the trigonometric root
//   p0 = a2^2/9 - a1/3, q0 = (a1 a2 - 3 a0)/6 - a2^3/27,
//   alpha = 2 sqrt(p0) cos( acos(q0 / p0^(3/2)) / 3 + 4 pi / 3 ) - a2/3
// with p0 and q0 collapsed algebraically (using m1+m2+m3 = 1) to
//   case (3): p0 = 2 m1 m2,                   q0 = 3/2 m1 m2 (m12 - 2 w m3)
//   case (4): p0 = m1 m2 - (m12 - m3)^2 / 4,  q0 = 3/4 m1 m2 m3 (1 - 2 w)
// -- the literal a2, a1, a0 arithmetic loses all significance in fp32 when m1 is small
// ("SZ cancellation").
// ---------------------------------------------------------------------------------------
template <>
struct Precise<SZ> {
    struct L1 {
        float S, m1, m2, m3;
    };
    static __device__ __forceinline__ L1 normalise(float n1, float n2, float n3) {
        L1 t;
        t.S = (n1 + n2) + n3;
        const float inv = Math<false>::div(1.0f, t.S);
        t.m1 = n1 * inv;
        t.m2 = n2 * inv;
        t.m3 = n3 * inv;
        return t;
    }
    static __device__ __forceinline__ float cheap(float n1, float n2, float n3, float V, int &kind) {
        const L1 t = normalise(n1, n2, n3);
        const float m12 = t.m1 + t.m2;
        const float W = 2.0f * V * t.m3;
        const float x = 3.0f * W * t.m2;                                   // 6 w m2 m3
        const float s1 = t.m1 * t.m1;                                      // w < v1 <=> x < m1^2
        const bool c5 = m12 <= W;                                          // (5)
        const bool c1 = x < s1;                                            // (1)
        const bool c2 = x <= fmaf(3.0f * t.m2, t.m2 - t.m1, s1);           // (2): v1 <= w <= v2
        const float a5 = fmaf(V, t.m3, 0.5f * m12);
        const float a2 = 0.5f * (t.m1 + Math<false>::sqrt(fmaxf(fmaf(4.0f * W, t.m2, -s1 * (1.0f / 3.0f)), 0.0f)));
        kind = c5 ? KIND_DONE : (c1 ? KIND_HEAVY_B : (c2 ? KIND_DONE : KIND_HEAVY_A));
        return __fmul_rn(c5 ? a5 : a2, t.S);
    }
    static __device__ __forceinline__ float heavy_a(float n1, float n2, float n3, float V) {
        typedef Math<false> M;
        const L1 t = normalise(n1, n2, n3);
        const float m1 = t.m1, m2 = t.m2, m3 = t.m3;
        const float m12 = m1 + m2;
        const float W = 2.0f * V * m3;
        const float x = 3.0f * W * m2;
        const float s1 = m1 * m1;
        const float q = m1 * m2;
        // 6 m1 m2 m3 v3 of Listing 3; case (4) iff m3 < m12 and w6 >= it
        float v3n = m3 * m3 * fmaf(3.0f, m12, -m3);
        v3n = fmaf(s1, fmaf(-3.0f, m3, m1), v3n);
        v3n = fmaf(m2 * m2, fmaf(-3.0f, m3, m2), v3n);
        const bool c4 = m3 < m12 && x * m1 >= v3n;
        const float em = m12 - m3;
        const float p0 = c4 ? fmaf(-0.25f * em, em, q) : q + q;
        const float q0 = c4 ? 0.75f * q * (m3 - W) : 1.5f * q * (m12 - W);
        const float sp = M::sqrt(p0);
        const float theta = M::acos(M::div(q0, p0 * sp)) * (1.0f / 3.0f);
        // cos(theta + 4 pi/3) evaluated as cos(theta - 2 pi/3): same angle, |arg| < pi
        float alpha = fmaf(2.0f * sp, M::cos(theta - 2.0943951f), c4 ? 0.5f : m12);
        alpha = fmaxf(alpha, c4 ? m3 : m2);                                // bracket floor; drops NaN
        return __fmul_rn(alpha, t.S);
    }
    static __device__ __forceinline__ float heavy_b(float n1, float n2, float n3, float V) {
        const L1 t = normalise(n1, n2, n3);
        const float w6 = 3.0f * (2.0f * V * t.m3) * t.m2 * t.m1;
        return __fmul_rn(Math<false>::cbrt(w6), t.S);                      // (1): cbrt(w6)
    }
};

// ---------------------------------------------------------------------------------------
// method 2: Newton-Raphson for cases (1), (3), (4); closed forms for (2), (5)  (sect. 2.5)
// Fixed, unrolled trip counts: case (1) on d^3 - 6 V n1 n2 n3 from the
// integer-arithmetic seed, cases (3)/(4) on the depressed cubics from the top of the bracket
// (tau0 = min(0, e) resp. 0), where F is decreasing and concave so the iteration is monotone.
// ---------------------------------------------------------------------------------------
template <>
struct Precise<NEWTON> : CheapN {
    static __device__ __forceinline__ float heavy_a(float n1, float n2, float n3, float V) {
        const Cubic34 c = cubic34(n1, n2, n3, V);
        const float tau = newton_cubic<false, 4>(c.p, c.r, c.hi);
        return fmaxf(__fadd_rn(c.base, tau), c.floor);
    }
    static __device__ __forceinline__ float heavy_b(float n1, float n2, float n3, float V) {
        const float k = k6(n1, n2, n3, V);                                 // (1)
        return newton_cubic<false, 3>(0.0f, k, cbrt_seed(k));
    }
};

// ---------------------------------------------------------------------------------------
// method 3: nested intervals (bisection) for cases (3), (4); closed forms otherwise (sect. 2.5)
// F is decreasing on the bracket [lo, hi] with F(lo) >= 0 >= F(hi).
// ---------------------------------------------------------------------------------------
// Precise: halve until the fp32 midpoint stops moving -- a data-dependent trip count that
// grows with the initial width, as the paper describes ("not unrolled").
__device__ __forceinline__ float bisect_cubic_converged(float p, float r, float lo, float hi) {
    for (int i = 0; i < 64; ++i) {
        const float mid = 0.5f * (lo + hi);
        if (!(mid > lo && mid < hi)) break;
        const float F = fmaf(fmaf(mid, mid, -p), mid, -r);
        if (F > 0.0f) lo = mid; else hi = mid;
    }
    return 0.5f * (lo + hi);
}

template <>
struct Precise<NESTED> : CheapN {
    static __device__ __forceinline__ float heavy_a(float n1, float n2, float n3, float V) {
        const Cubic34 c = cubic34(n1, n2, n3, V);
        const float tau = bisect_cubic_converged(c.p, c.r, c.lo, c.hi);
        return fmaxf(__fadd_rn(c.base, tau), c.floor);
    }
    static __device__ __forceinline__ float heavy_b(float n1, float n2, float n3, float V) {
        return Math<false>::cbrt(k6(n1, n2, n3, V));                       // (1)
    }
};

template <int METHOD, bool FAST>
struct Solver;

// scalar form of the four precise methods: branches in the paper's order (5)->(2)->(1)->(3)->(4)
template <int METHOD>
struct Solver<METHOD, false> {
    static __device__ __forceinline__ float reduced_offset(float n1, float n2, float n3, float V) {
        int kind;
        float d = Precise<METHOD>::cheap(n1, n2, n3, V, kind);             // (5), (2)
        if (kind == KIND_HEAVY_B) d = Precise<METHOD>::heavy_b(n1, n2, n3, V);        // (1)
        else if (kind == KIND_HEAVY_A) d = Precise<METHOD>::heavy_a(n1, n2, n3, V);   // (3), (4)
        return d;
    }
};

// ---------------------------------------------------------------------------------------
// method 4: the SZ solution as implemented by Kawano, "translated ... without further
// optimization" -- Listing 3, kept for the paper's five-way comparison and
// for its documented defect: for n = (1,0,0) and V0 in {0, 1} it returns NaN (PAPER.md:217,
// 256), which is why Tables 1-3 show E_avg = -NaN for it.  NOT edge-case complete and NOT
// cancellation free (its a2, a1, a0 arithmetic loses the digits of a small m1): use SZ.
//
// The listing is truncated in PAPER.md; the surviving lines are followed literally (thresholds
// v1, v1 + (vm2-vm1)/(2 vm3), v3; cases (1), (2), (5) closed forms; a2, a1, a0 of cases (3)/(4);
// the 4/3 pi constant; return l*copysign(0.5-alpha, V0-0.5)), the lost ones are filled in from
// the text (R21): vm_i = n_i / l with the L1 norm l, w = V, w6 =
// 6 vm1 vm2 vm3 w, v1 = vm1^2 / (6 vm2 vm3 + tiny) with tiny = 1e-30 ("a tiny constant to the
// denominator"), v3 = its cubic form if vm3 < vm12 else vm12 / (2 vm3)
// with case (5) taken only in the latter situation, and the textbook trigonometric root of alpha^3 + a2 alpha^2 + a1 alpha + a0:
// p0 = a2^2/9 - a1/3, q0 = (a1 a2 - 3 a0)/6 - a2^3/27, theta = acos(q0 / sqrt(p0^3)) / 3,
// alpha = 2 sqrt(p0) cos(theta + 4/3 pi) - a2/3.
// ---------------------------------------------------------------------------------------
template <>
struct Solver<KAWANO, false> {
    static __device__ __forceinline__ float reduced_offset(float n1, float n2, float n3, float V) {
        const float l = (n1 + n2) + n3;
        const float vm1 = n1 / l, vm2 = n2 / l, vm3 = n3 / l, vm12 = vm1 + vm2;
        const float w = V;
        const float w6 = 6.0f * vm1 * vm2 * vm3 * w;
        const float v1 = vm1 * vm1 / (6.0f * vm2 * vm3 + 1e-30f);
        float alpha = 0.0f;
        if (w < v1) {
            alpha = cbrtf(w6);                                                         // case (1)
        } else if (w < v1 + 0.5f * (vm2 - vm1) / vm3) {
            alpha = 0.5f * (vm1 + sqrtf(vm1 * vm1 + 8.0f * vm2 * vm3 * (w - v1)));     // case (2)
        } else {
            const float v3 = vm3 < vm12
                ? (vm3 * vm3 * (3.0f * vm12 - vm3) + vm1 * vm1 * (vm1 - 3.0f * vm3) +
                   vm2 * vm2 * (vm2 - 3.0f * vm3)) / (6.0f * vm1 * vm2 * vm3)
                : 0.5f * vm12 / vm3;
            // case (5) exists only for vm12 <= vm3 (with vm3 < vm12, w >= v3 is case (4))
            if (vm12 <= vm3 && v3 <= w) alpha = vm3 * w + 0.5f * vm12;
            if (alpha == 0.0f) {
                float a0, a1, a2;
                if (w < v3) {                                                          // case (3)
                    a2 = -3.0f * vm12;
                    a1 = 3.0f * (vm1 * vm1 + vm2 * vm2);
                    a0 = w6 - vm1 * vm1 * vm1 - vm2 * vm2 * vm2;
                } else {                                                               // case (4)
                    a2 = -1.5f;
                    a1 = 1.5f * (vm1 * vm1 + vm2 * vm2 + vm3 * vm3);
                    a0 = 0.5f * (w6 - vm1 * vm1 * vm1 - vm2 * vm2 * vm2 - vm3 * vm3 * vm3);
                }
                const float p0 = a2 * a2 * (1.0f / 9.0f) - a1 * (1.0f / 3.0f);
                const float q0 = (a1 * a2 - 3.0f * a0) * (1.0f / 6.0f) - a2 * a2 * a2 * (1.0f / 27.0f);
                const float theta = acosf(q0 / sqrtf(p0 * p0 * p0)) * (1.0f / 3.0f);
                alpha = 2.0f * sqrtf(p0) * cosf(theta + 4.1887902f) - a2 * (1.0f / 3.0f);   // 4/3 pi
            }
        }
        return alpha * l;
    }
};

// ---------------------------------------------------------------------------------------
// frame: symmetry reduction (eq. (2)-(5)) -> method -> sign restore (eq. (8))
// ---------------------------------------------------------------------------------------
struct Reduced {
    float n1, n2, n3, V;
};
__device__ __forceinline__ Reduced reduce_cell(float V0, float nx, float ny, float nz) {
    const float a = fabsf(nx), b = fabsf(ny), c = fabsf(nz);
    Reduced r;
    r.n1 = min3(a, b, c);                                              // eq. (2)
    r.n3 = max3(a, b, c);                                              // eq. (3)
    r.n2 = fmaxf(fminf(a, b), fminf(fmaxf(a, b), c));                  // eq. (4): the median
    // eq. (5): 1/2 - |V0 - 1/2| = min(V0, 1 - V0), which is exact in fp32 for V0 in [0,1]
    r.V = fmaxf(fminf(V0, 1.0f - V0), 0.0f);
    return r;
}
__device__ __forceinline__ float half_l1(const Reduced &c) { return 0.5f * ((c.n1 + c.n2) + c.n3); }   // S/2
// d0 = sign(V0 - 1/2) (S/2 - d), eq. (8), with d clamped to [0, S/2] (drops a NaN)
template <bool CLAMP>
__device__ __forceinline__ float restore_cell(float V0, float hS, float d) {
    if (CLAMP) d = fminf(fmaxf(d, 0.0f), hS);
    const float r = __fsub_rn(hS, d);
    return V0 > 0.5f ? r : -r;
}

template <int METHOD, bool FAST>
__device__ __forceinline__ float solve_cell(float V0, float nx, float ny, float nz) {
    const Reduced c = reduce_cell(V0, nx, ny, nz);
    const float d = Solver<METHOD, FAST>::reduced_offset(c.n1, c.n2, c.n3, c.V);
    return restore_cell<METHOD != KAWANO>(V0, half_l1(c), d);          // Listing 3 has no clamp: its NaN is kept
}

}  // namespace plic
