"""Derives the polynomial coefficients hard-coded in plic_packed.cuh (run by hand; prints them).

  neg_sin_third_asin_fast2: g(C) = sin(asin(C)/3) ~ C * P3(C^2) on [0, 0.9], then one Newton step
                        on 3g - 4g^3 = C.
  acos_fast2:           acos(x) ~ sqrt(1-x) * Q(x) on [0, 1].

Weighted least squares on Chebyshev nodes with Lawson re-weighting (converges to the minimax
fit).  Part of the CUDA path's sources; nothing under oracle/ or tests/ uses it.
"""
import numpy as np


def lawson(A, y, iters=200):
    w = np.ones(len(y))
    for _ in range(iters):
        co, *_ = np.linalg.lstsq(A * w[:, None], y * w, rcond=None)
        r = np.abs(A @ co - y)
        w = w * np.sqrt((r + 1e-300) / (r.max() + 1e-300))
        w /= w.max()
    return co, np.abs(A @ co - y).max()


def main():
    t = np.cos(np.linspace(0.0, np.pi, 8001))
    # --- g(C) on [0, 0.9] ---------------------------------------------------------------
    C = 0.45 * (t + 1.0)
    g = np.sin(np.arcsin(C) / 3.0)
    for ncoef in (3, 4):
        A = np.stack([C ** (2 * k + 1) for k in range(ncoef)], 1)
        co, e0 = lawson(A, g)
        g0 = (A @ co).astype(np.float32).astype(np.float64)
        g1 = (C - 8 * g0 ** 3) / (3 - 12 * g0 ** 2)
        print("sin_third_asin ncoef=%d start err %.3e, after Newton %.3e" % (ncoef, e0, np.abs(g1 - g).max()))
        print("   ", ", ".join("%.9gf" % c for c in co))
    # --- acos(x) = sqrt(1-x) Q(x) on [0, 1] ------------------------------------------------
    x = 0.5 * (t + 1.0)
    x = x[x < 1.0]
    y = np.arccos(x) / np.sqrt(1.0 - x)
    for deg in (3, 4, 5, 7):
        A = np.stack([x ** k for k in range(deg + 1)], 1)
        co, e = lawson(A, y)
        err = np.abs(np.sqrt(1 - x) * (A @ co) - np.arccos(x)).max()
        print("acos deg=%d ratio err %.3e, acos err %.3e" % (deg, e, err))
        print("   ", ", ".join("%.10gf" % c for c in co))


if __name__ == "__main__":
    main()
