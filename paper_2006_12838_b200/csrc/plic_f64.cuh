// plic_f64.cuh -- the four methods in fp64 arithmetic (plic_solve_f64, include/plic.h).
//
// The paper fixes fp32 ("floating-point precision ... 32-bit"); SURVEY.md 8f row f4
// asks for an fp64 variant as a "next" row: 40 B per cell instead of 20, IEEE division and square
// root, CUDA libm cbrt / asin / sin / acos / cos in double precision.  It is the like-for-like GPU
// counterpart of the fp64 bisection oracle.  Same formulation as the precise fp32 kernels
// (plic_methods.cuh): a-priori case selection (eq. (26), misprint corrected), depressed cubics for
// cases (3)/(4), the three pieces cheap() / heavy_a() / heavy_b() evaluated by map_compact in dense
// warps.  Only the trip counts differ: Newton-Raphson needs 7 (cases (3)/(4)) and 6 (case (1)) steps
// to reach fp64 rounding from the same start values (quadratic convergence: fp32's 4 steps leave
// ~1e-11), nested intervals halves until the fp64 midpoint stops moving (~50 halvings).
#pragma once
#include "plic_methods.cuh"

namespace plic {
namespace f64 {

__device__ __forceinline__ bool is_case4(double q, double e, double ee, double z) {
    const double h = fma(fma(-6.0, q, ee), e, -3.0 * (q * z));
    return (e < 0.0) && (h > 0.0);
}

// cases (5), (2) and the case decision, as CheapN in plic_methods.cuh
struct CheapN {
    static __device__ __forceinline__ double cheap(double n1, double n2, double n3, double V, int &kind) {
        const double n12 = n1 + n2;
        const double W = 2.0 * V * n3;
        const double x = 3.0 * W * n2;                                     // 6 V n2 n3
        const double s1 = n1 * n1;
        const bool c5 = n12 <= W;                                          // (5) eq. (26)
        const bool c1 = x < s1;                                            // (1)
        const bool c2 = x <= fma(3.0 * n2, n2 - n1, s1);                   // (2), misprint corrected
        const double d5 = fma(V, n3, 0.5 * n12);
        const double d2 = fma(0.5, n1, sqrt(fmax(fma(W, n2, -s1 * (1.0 / 12.0)), 0.0)));
        kind = c5 ? KIND_DONE : (c1 ? KIND_HEAVY_B : (c2 ? KIND_DONE : KIND_HEAVY_A));
        return c5 ? d5 : d2;
    }
    static __device__ __forceinline__ double k6(double n1, double n2, double n3, double V) {
        return __dmul_rn(3.0 * (2.0 * V * n3) * n2, n1);                   // 6 V n1 n2 n3
    }
};

struct Cubic34 {
    double p, r, lo, hi, base, floor;
};
__device__ __forceinline__ Cubic34 cubic34(double n1, double n2, double n3, double V) {
    const double n12 = n1 + n2;
    const double W = 2.0 * V * n3;
    const double q = n1 * n2;
    const double e = n3 - n12;
    const double z = n12 - W;
    const double ee = e * e;
    const bool c4 = is_case4(q, e, ee, z);
    const double hS = 0.5 * (n12 + n3);
    Cubic34 c;
    c.p = c4 ? 0.75 * fma(4.0, q, -ee) : 6.0 * q;
    c.r = c4 ? 1.5 * q * (n3 - W) : 3.0 * q * z;
    c.lo = c4 ? n3 - hS : -n1;
    c.hi = c4 ? 0.0 : fmin(e, 0.0);
    c.base = c4 ? hS : n12;
    c.floor = c4 ? n3 : n2;
    return c;
}

template <int ITERS>
__device__ __forceinline__ double newton_cubic(double p, double r, double tau) {
#pragma unroll
    for (int i = 0; i < ITERS; ++i) {
        const double t2 = tau * tau;
        tau = fma(2.0 * t2, tau, r) / fma(3.0, t2, -p);
    }
    return tau;
}

// start value for the cube root: exponent / 3 on the high word (relative error < 4 %)
__device__ __forceinline__ double cbrt_seed(double k) {
    return __hiloint2double(__double2hiint(k) / 3 + 715094163, 0);
}

__device__ __forceinline__ double bisect_cubic_converged(double p, double r, double lo, double hi) {
    for (int i = 0; i < 128; ++i) {
        const double mid = 0.5 * (lo + hi);
        if (!(mid > lo && mid < hi)) break;
        const double F = fma(fma(mid, mid, -p), mid, -r);
        if (F > 0.0) lo = mid; else hi = mid;
    }
    return 0.5 * (lo + hi);
}

template <int METHOD>
struct Precise;

// method 0: analytic inverse, eq. (25)/(26), one trigonometric evaluation for (3)/(4)
template <>
struct Precise<ANALYTIC> : CheapN {
    static __device__ __forceinline__ double heavy_a(double n1, double n2, double n3, double V) {
        const double n12 = n1 + n2;
        const double W = 2.0 * V * n3;
        const double q = n1 * n2;
        const double e = n3 - n12;
        const double z = n12 - W;
        const double ee = e * e;
        const bool c4 = is_case4(q, e, ee, z);
        const double A = c4 ? fma(4.0, q, -ee) : q + q;                    // u or 2 q
        const double sA = sqrt(A);
        const double num = c4 ? 6.0 * q * (n3 - W) : 0.75 * z;
        const double C = num / (c4 ? A * sA : sA);
        const double amp = c4 ? -sA : -2.0 * sA;
        const double d = fma(amp, sin(asin(fmin(C, 1.0)) * (1.0 / 3.0)), c4 ? 0.5 * (n12 + n3) : n12);
        return fmax(d, c4 ? n3 : n2);                                      // bracket floor; drops NaN
    }
    static __device__ __forceinline__ double heavy_b(double n1, double n2, double n3, double V) {
        return cbrt(k6(n1, n2, n3, V));                                    // (1)
    }
};

// method 1: Scardovelli-Zaleski (sect. 2.4), L1-normalised, collapsed p0, q0
template <>
struct Precise<SZ> {
    struct L1 {
        double S, m1, m2, m3;
    };
    static __device__ __forceinline__ L1 normalise(double n1, double n2, double n3) {
        L1 t;
        t.S = (n1 + n2) + n3;
        const double inv = 1.0 / t.S;
        t.m1 = n1 * inv;
        t.m2 = n2 * inv;
        t.m3 = n3 * inv;
        return t;
    }
    static __device__ __forceinline__ double cheap(double n1, double n2, double n3, double V, int &kind) {
        const L1 t = normalise(n1, n2, n3);
        const double m12 = t.m1 + t.m2;
        const double W = 2.0 * V * t.m3;
        const double x = 3.0 * W * t.m2;
        const double s1 = t.m1 * t.m1;
        const bool c5 = m12 <= W;
        const bool c1 = x < s1;
        const bool c2 = x <= fma(3.0 * t.m2, t.m2 - t.m1, s1);
        const double a5 = fma(V, t.m3, 0.5 * m12);
        const double a2 = 0.5 * (t.m1 + sqrt(fmax(fma(4.0 * W, t.m2, -s1 * (1.0 / 3.0)), 0.0)));
        kind = c5 ? KIND_DONE : (c1 ? KIND_HEAVY_B : (c2 ? KIND_DONE : KIND_HEAVY_A));
        return __dmul_rn(c5 ? a5 : a2, t.S);
    }
    static __device__ __forceinline__ double heavy_a(double n1, double n2, double n3, double V) {
        const L1 t = normalise(n1, n2, n3);
        const double m1 = t.m1, m2 = t.m2, m3 = t.m3;
        const double m12 = m1 + m2;
        const double W = 2.0 * V * m3;
        const double x = 3.0 * W * m2;
        const double s1 = m1 * m1;
        const double q = m1 * m2;
        double v3n = m3 * m3 * fma(3.0, m12, -m3);                         // 6 m1 m2 m3 v3
        v3n = fma(s1, fma(-3.0, m3, m1), v3n);
        v3n = fma(m2 * m2, fma(-3.0, m3, m2), v3n);
        const bool c4 = m3 < m12 && x * m1 >= v3n;
        const double em = m12 - m3;
        const double p0 = c4 ? fma(-0.25 * em, em, q) : q + q;
        const double q0 = c4 ? 0.75 * q * (m3 - W) : 1.5 * q * (m12 - W);
        const double sp = sqrt(p0);
        const double theta = acos(fmin(q0 / (p0 * sp), 1.0)) * (1.0 / 3.0);
        double alpha = fma(2.0 * sp, cos(theta - 2.0943951023931954923), c4 ? 0.5 : m12);
        alpha = fmax(alpha, c4 ? m3 : m2);                                 // bracket floor; drops NaN
        return __dmul_rn(alpha, t.S);
    }
    static __device__ __forceinline__ double heavy_b(double n1, double n2, double n3, double V) {
        const L1 t = normalise(n1, n2, n3);
        const double w6 = 3.0 * (2.0 * V * t.m3) * t.m2 * t.m1;
        return __dmul_rn(cbrt(w6), t.S);
    }
};

// method 2: Newton-Raphson (sect. 2.5), fixed trip counts
template <>
struct Precise<NEWTON> : CheapN {
    static __device__ __forceinline__ double heavy_a(double n1, double n2, double n3, double V) {
        const Cubic34 c = cubic34(n1, n2, n3, V);
        const double tau = newton_cubic<7>(c.p, c.r, c.hi);
        return fmax(__dadd_rn(c.base, tau), c.floor);
    }
    static __device__ __forceinline__ double heavy_b(double n1, double n2, double n3, double V) {
        const double k = k6(n1, n2, n3, V);
        return newton_cubic<6>(0.0, k, cbrt_seed(k));
    }
};

// method 3: nested intervals (sect. 2.5), until the fp64 midpoint stops moving
template <>
struct Precise<NESTED> : CheapN {
    static __device__ __forceinline__ double heavy_a(double n1, double n2, double n3, double V) {
        const Cubic34 c = cubic34(n1, n2, n3, V);
        const double tau = bisect_cubic_converged(c.p, c.r, c.lo, c.hi);
        return fmax(__dadd_rn(c.base, tau), c.floor);
    }
    static __device__ __forceinline__ double heavy_b(double n1, double n2, double n3, double V) {
        return cbrt(k6(n1, n2, n3, V));
    }
};

// frame: eq. (2)-(5) in, eq. (8) out
struct Reduced {
    double n1, n2, n3, V;
};
__device__ __forceinline__ Reduced reduce_cell(double V0, double nx, double ny, double nz) {
    const double a = fabs(nx), b = fabs(ny), c = fabs(nz);
    Reduced r;
    r.n1 = fmin(fmin(a, b), c);                                        // eq. (2)
    r.n3 = fmax(fmax(a, b), c);                                        // eq. (3)
    r.n2 = fmax(fmin(a, b), fmin(fmax(a, b), c));                      // eq. (4): the median
    r.V = fmax(fmin(V0, 1.0 - V0), 0.0);                               // eq. (5)
    return r;
}
__device__ __forceinline__ double half_l1(const Reduced &c) { return 0.5 * ((c.n1 + c.n2) + c.n3); }
__device__ __forceinline__ double restore_cell(double V0, double hS, double d) {
    d = fmin(fmax(d, 0.0), hS);
    const double r = __dsub_rn(hS, d);
    return V0 > 0.5 ? r : -r;                                          // eq. (8)
}

template <int METHOD>
__device__ __forceinline__ double solve_cell(double V0, double nx, double ny, double nz) {
    const Reduced c = reduce_cell(V0, nx, ny, nz);
    int kind;
    double d = Precise<METHOD>::cheap(c.n1, c.n2, c.n3, c.V, kind);
    if (kind == KIND_HEAVY_B) d = Precise<METHOD>::heavy_b(c.n1, c.n2, c.n3, c.V);
    else if (kind == KIND_HEAVY_A) d = Precise<METHOD>::heavy_a(c.n1, c.n2, c.n3, c.V);
    return restore_cell(V0, half_l1(c), d);
}

}  // namespace f64
}  // namespace plic
