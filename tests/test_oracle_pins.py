"""Pins for the fp64 oracle (oracle/plic_oracle.c) against things other than itself.

Each test checks the oracle against what the paper or elementary mathematics fixes:
closed forms of the paper's cases (1), (2), (5) (eq. (25)), the 1D/2D
special cases (eq. (28), (30)), symmetry / monotonicity
(PAPER.md:48), the endpoints of eq. (1), invariance under the mirror
and sort of eq. (2)-(4), the textbook inclusion-exclusion volume of a box cut by a
half-space (no case split), brute-force quadrature of the definition
Vol{x in cube : n.x <= d0}, the vertex-count definition of the five cases (fig. 1),
and hand-derived worked examples (tests/golden/worked_examples.txt).
"""
import itertools
import math
import os

import numpy as np
import pytest

import oracle

HERE = os.path.dirname(os.path.abspath(__file__))
RNG = np.random.default_rng(20061283)


def unit(g):
    g = np.asarray(g, dtype=np.float64)
    return g / np.linalg.norm(g, axis=-1, keepdims=True)


def sorted_abs(n):
    return np.sort(np.abs(n), axis=-1)


# ----------------------------------------------------------------------------------
# textbook formula: volume of [0,1]^k cut by a.x <= t, a_i > 0 (inclusion-exclusion)
# ----------------------------------------------------------------------------------
def box_cut_volume(a, t):
    a = [x for x in a if x > 0.0]
    k = len(a)
    if k == 0:
        return 1.0 if t >= 0 else 0.0
    tot = 0.0
    for v in itertools.product((0, 1), repeat=k):
        r = t - sum(ai for ai, vi in zip(a, v) if vi)
        if r > 0.0:
            tot += (-1) ** sum(v) * r ** k
    return tot / (math.factorial(k) * math.prod(a))


def test_p11_inclusion_exclusion_3d():
    n = unit(RNG.standard_normal((3000, 3)))
    S = np.abs(n).sum(1)
    d0 = (RNG.random(3000) - 0.5) * S * 1.02      # a few planes miss the cube
    got = oracle.volume(d0, n[:, 0], n[:, 1], n[:, 2])
    ref = np.array([box_cut_volume(np.abs(ni), di + 0.5 * si) for ni, di, si in zip(n, d0, S)])
    ref = np.clip(ref, 0.0, 1.0)
    assert np.max(np.abs(got - ref)) < 5e-12


def test_p11_inclusion_exclusion_2d_1d():
    g = RNG.standard_normal((1000, 3))
    g[:, 1] = 0.0                                  # 2D normals, exact zero component
    n = unit(g)
    S = np.abs(n).sum(1)
    d0 = (RNG.random(1000) - 0.5) * S
    got = oracle.volume(d0, n[:, 0], n[:, 1], n[:, 2])
    ref = np.array([box_cut_volume(np.abs(ni), di + 0.5 * si) for ni, di, si in zip(n, d0, S)])
    assert np.max(np.abs(got - ref)) < 1e-13
    for axis in range(3):                          # 1D: V0 = d0 + 1/2
        e = np.zeros(3)
        e[axis] = -1.0
        d = np.linspace(-0.5, 0.5, 41)
        assert np.max(np.abs(oracle.volume(d, *e) - (d + 0.5))) < 1e-15


# ----------------------------------------------------------------------------------
# brute force on the definition
# ----------------------------------------------------------------------------------
def column_quadrature(n, d0, m=1500):
    """Vol{x in [-1/2,1/2]^3 : n.x <= d0} by integrating the height of each (u,v)
    column along the axis of the largest |n| component (midpoint rule, m^2 columns)."""
    n = np.asarray(n, dtype=np.float64)
    k = int(np.argmax(np.abs(n)))
    o = [i for i in range(3) if i != k]
    g = (np.arange(m) + 0.5) / m - 0.5
    u, v = np.meshgrid(g, g, indexing="ij")
    w = (d0 - n[o[0]] * u - n[o[1]] * v) / n[k]    # plane height along axis k
    if n[k] > 0:                                   # region is  x_k <= w
        h = np.clip(w + 0.5, 0.0, 1.0)
    else:                                          # region is  x_k >= w
        h = np.clip(0.5 - w, 0.0, 1.0)
    return float(h.mean())


def test_p12_column_quadrature_signed_normals():
    n = unit(RNG.standard_normal((24, 3)))
    n[0] = unit([1e-3, -0.4, 0.9])
    n[1] = unit([-0.5, 0.5, 0.70710678])
    S = np.abs(n).sum(1)
    d0 = (RNG.random(24) - 0.5) * S
    got = oracle.volume(d0, n[:, 0], n[:, 1], n[:, 2])
    ref = np.array([column_quadrature(ni, di) for ni, di in zip(n, d0)])
    assert np.max(np.abs(got - ref)) < 2e-6


def test_p12_point_counting_direction_of_normal():
    # coarse 3-D point count; pins which side of the plane is counted (reading R4)
    m = 60
    g = (np.arange(m) + 0.5) / m - 0.5
    X, Y, Z = np.meshgrid(g, g, g, indexing="ij")
    for n, d0 in [((0.0, 0.0, 1.0), 0.25), ((0.0, 0.0, -1.0), 0.25),
                  (unit([1.0, -2.0, 0.5]), -0.3), (unit([-1.0, -1.0, -1.0]), 0.4)]:
        frac = np.mean(n[0] * X + n[1] * Y + n[2] * Z <= d0)
        assert abs(float(oracle.volume(d0, *n)) - frac) < 6e-3


# ----------------------------------------------------------------------------------
# the five cases by vertex count (fig. 1)
# ----------------------------------------------------------------------------------
def test_case_is_vertex_configuration():
    n = unit(RNG.standard_normal((4000, 3)))
    a = sorted_abs(n)
    S = a.sum(1)
    d = RNG.random(4000) * 0.5 * S                 # reduced offset from the corner
    d0 = d - 0.5 * S
    kase = oracle.case(d0, n[:, 0], n[:, 1], n[:, 2])
    for ai, di, ki in zip(a, d, kase):
        below = {v for v in itertools.product((0, 1), repeat=3)
                 if sum(x * y for x, y in zip(ai, v)) < di}
        nb = len(below)
        if ki == 1:
            assert below <= {(0, 0, 0)}
        elif ki == 2:
            assert below == {(0, 0, 0), (1, 0, 0)} or nb == 1  # d == n1 tie
        elif ki == 3:
            assert below == {(0, 0, 0), (1, 0, 0), (0, 1, 0)}
        elif ki == 4:
            assert below == {(0, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1)}
        else:
            assert ki == 5
            assert below == {(0, 0, 0), (1, 0, 0), (0, 1, 0), (1, 1, 0)}
    frac = np.bincount(kase, minlength=6)[1:] / 4000.0
    assert (frac > 0.02).all()                     # every case is exercised


# ----------------------------------------------------------------------------------
# closed forms of eq. (25): cases (1), (2), (5)
# ----------------------------------------------------------------------------------
def _random_sorted(nrows):
    n = unit(RNG.standard_normal((nrows, 3)))
    a = sorted_abs(n)
    return n, a[:, 0], a[:, 1], a[:, 2]


def test_p1_case1_closed_form():
    n, n1, n2, n3 = _random_sorted(5000)
    Vmax = n1 ** 2 / (6 * n2 * n3)                 # V(d = n1), eq. (11) case (1)
    V = RNG.random(5000) * np.minimum(Vmax, 0.5)
    d = np.cbrt(6 * V * n1 * n2 * n3)              # eq. (25) case (1)
    S = n1 + n2 + n3
    for V0, d0 in ((V, -(0.5 * S - d)), (1 - V, 0.5 * S - d)):     # eq. (8)
        got = oracle.solve(V0, n[:, 0], n[:, 1], n[:, 2])
        assert np.max(np.abs(got - d0)) < 1e-9


def test_p2_case2_closed_form():
    n, n1, n2, n3 = _random_sorted(5000)
    Vlo = n1 ** 2 / (6 * n2 * n3)                                  # V(d = n1)
    Vhi = (3 * n2 ** 2 - 3 * n2 * n1 + n1 ** 2) / (6 * n2 * n3)    # V(d = n2), eq. (11) case (2)
    V = Vlo + RNG.random(5000) * (np.minimum(Vhi, 0.5) - Vlo)
    ok = V <= 0.5
    d = 0.5 * n1 + np.sqrt(2 * V * n2 * n3 - n1 ** 2 / 12)         # eq. (25) case (2)
    S = n1 + n2 + n3
    got = oracle.solve(V, n[:, 0], n[:, 1], n[:, 2])
    assert ok.sum() > 4000
    assert np.max(np.abs(got - (d - 0.5 * S))[ok]) < 1e-11
    got = oracle.solve(1 - V, n[:, 0], n[:, 1], n[:, 2])
    assert np.max(np.abs(got - (0.5 * S - d))[ok]) < 1e-9


def test_p3_case5_closed_form():
    n, n1, n2, n3 = _random_sorted(20000)
    sel = n1 + n2 < n3                              # case (5) has non-zero width
    n, n1, n2, n3 = n[sel], n1[sel], n2[sel], n3[sel]
    assert sel.sum() > 2000
    Vlo = (n1 + n2) / (2 * n3)                      # eq. (26) case (5):  n1+n2 <= 2 V n3
    V = Vlo + RNG.random(n1.shape[0]) * (0.5 - Vlo)
    d = V * n3 + 0.5 * (n1 + n2)                    # eq. (25) case (5)
    S = n1 + n2 + n3
    got = oracle.solve(V, n[:, 0], n[:, 1], n[:, 2])
    assert np.max(np.abs(got - (d - 0.5 * S))) < 1e-12


def test_p4_axis_aligned():
    V0 = np.concatenate([np.linspace(0, 1, 101), [1e-7, 1 - 1e-7, 0.5]])
    for axis in range(3):
        for s in (1.0, -1.0):
            e = np.zeros(3)
            e[axis] = s
            got = oracle.solve(V0, *e)
            assert np.max(np.abs(got - (V0 - 0.5))) < 1e-13      # eq. (28)


def test_p5_two_dimensional():
    g = RNG.standard_normal((3000, 3))
    zero_axis = RNG.integers(0, 3, 3000)
    g[np.arange(3000), zero_axis] = 0.0
    n = unit(g)
    a = sorted_abs(n)
    n2, n3 = a[:, 1], a[:, 2]
    V = RNG.random(3000) * 0.5
    d = np.where(2 * V * n3 <= n2, np.sqrt(2 * V * n2 * n3), V * n3 + 0.5 * n2)   # eq. (30)
    got = oracle.solve(V, n[:, 0], n[:, 1], n[:, 2])
    assert np.max(np.abs(got - (d - 0.5 * (n2 + n3)))) < 1e-9


# ----------------------------------------------------------------------------------
# invariants
# ----------------------------------------------------------------------------------
def test_p6_symmetry():
    n = unit(RNG.standard_normal((4000, 3)))
    S = np.abs(n).sum(1)
    d0 = (RNG.random(4000) - 0.5) * S
    v = oracle.volume(d0, n[:, 0], n[:, 1], n[:, 2])
    vm = oracle.volume(-d0, n[:, 0], n[:, 1], n[:, 2])
    assert np.max(np.abs(v + vm - 1.0)) < 1e-15
    V0 = RNG.random(4000)
    a = oracle.solve(V0, n[:, 0], n[:, 1], n[:, 2])
    b = oracle.solve(1.0 - V0, n[:, 0], n[:, 1], n[:, 2])
    assert np.max(np.abs(a + b)) < 1e-12


def test_p7_monotone_and_continuous():
    normals = list(unit(RNG.standard_normal((40, 3))))
    normals += [unit([1, 1, 1]), unit([1, 1, 0]), unit([0, 0, 1]), unit([1, 2, 3]),
                unit([1e-6, 1, 1]), unit([1e-3, 2e-3, 1]), unit([0.5, 0.5, 0.7071])]
    for n in normals:
        S = np.abs(n).sum()
        d0 = np.linspace(-0.5 * S, 0.5 * S, 20001)
        v = oracle.volume(d0, *n)
        dv = np.diff(v)
        assert (dv >= -1e-15).all()
        # |dV/dd0| is the cross-section area <= sqrt(3) (central hexagon is 3*sqrt(3)/4)
        assert dv.max() <= 1.75 * (d0[1] - d0[0])
        a = np.sort(np.abs(n))
        for b in (a[0], a[1], a[2], a[0] + a[1]):   # continuity at every case boundary
            if b <= 0.5 * S:
                lo = oracle.volume(-(0.5 * S - b) - 1e-12, *n)
                hi = oracle.volume(-(0.5 * S - b) + 1e-12, *n)
                # eq. (11) cases (3)/(4) subtract cubes: fp64 noise ~ eps d^3 / (6 n1 n2 n3)
                noise = 2e-16 / (6 * a[0] * a[1] * a[2]) if a[0] > 0 else 0.0
                assert abs(hi - lo) < 1e-11 + noise


def test_p8_endpoints():
    n = unit(RNG.standard_normal((1000, 3)))
    S = np.abs(n).sum(1)
    assert (S >= 1.0 - 1e-12).all() and (S <= math.sqrt(3) + 1e-12).all()
    lo = oracle.solve(np.zeros(1000), n[:, 0], n[:, 1], n[:, 2])
    hi = oracle.solve(np.ones(1000), n[:, 0], n[:, 1], n[:, 2])
    assert np.max(np.abs(lo + 0.5 * S)) < 1e-15 and np.max(np.abs(hi - 0.5 * S)) < 1e-15
    assert np.array_equal(lo, -hi)
    assert np.max(np.abs(oracle.volume(lo, n[:, 0], n[:, 1], n[:, 2]))) == 0.0
    assert np.max(np.abs(oracle.volume(hi, n[:, 0], n[:, 1], n[:, 2]) - 1.0)) == 0.0
    # planes that miss the cube
    assert np.all(oracle.volume(-0.5 * S - 0.1, n[:, 0], n[:, 1], n[:, 2]) == 0.0)
    assert np.all(oracle.volume(0.5 * S + 0.1, n[:, 0], n[:, 1], n[:, 2]) == 1.0)
    # V0 just inside the ends stays inside the interval and close to the end
    d = oracle.solve(np.full(1000, 1e-30), n[:, 0], n[:, 1], n[:, 2])
    assert np.all(d >= lo) and np.all(d < lo + 1e-9)


def test_p9_permutation_and_sign_invariance():
    n = unit(RNG.standard_normal((500, 3)))
    V0 = RNG.random(500)
    ref = oracle.solve(V0, n[:, 0], n[:, 1], n[:, 2])
    for perm in itertools.permutations(range(3)):
        for sg in itertools.product((1.0, -1.0), repeat=3):
            m = n[:, perm] * np.asarray(sg)
            got = oracle.solve(V0, m[:, 0], m[:, 1], m[:, 2])
            assert np.max(np.abs(got - ref)) < 1e-13


def test_p10_homogeneity_of_forward_map():
    n = unit(RNG.standard_normal((500, 3)))
    d0 = (RNG.random(500) - 0.5) * np.abs(n).sum(1)
    ref = oracle.volume(d0, n[:, 0], n[:, 1], n[:, 2])
    for lam in (0.25, 3.0):
        got = oracle.volume(lam * d0, lam * n[:, 0], lam * n[:, 1], lam * n[:, 2])
        assert np.max(np.abs(got - ref)) < 1e-13


def test_p14_round_trip():
    n = unit(RNG.standard_normal((20000, 3)))
    V0 = RNG.random(20000)
    d0 = oracle.solve(V0, n[:, 0], n[:, 1], n[:, 2])
    back = oracle.volume(d0, n[:, 0], n[:, 1], n[:, 2])
    assert np.max(np.abs(back - V0)) < 2e-13
    assert np.all(np.abs(d0) <= 0.5 * np.abs(n).sum(1))


def test_exact_rational_check_small_n1():
    """eq. (11) subtracts cubes in cases (3)/(4); for a tiny smallest component the fp64
    rounding noise of V is ~ eps d^3/(6 n1 n2 n3), confined to the window of width n1 in
    d where those cases apply.  Check the oracle against the inclusion-exclusion formula
    in exact rational arithmetic: V stays within that noise model and the offset error
    min(n1, noise) stays below 1e-8, three orders under the 2e-5 parity tolerance."""
    from fractions import Fraction as F
    worst_v, worst_d = 0.0, 0.0
    for n1 in (1e-2, 1e-4, 1e-6, 1e-8, 3e-9, 1e-9, 1e-10, 1e-12):
        n = unit([n1, 0.6, 0.8])
        a = np.sort(np.abs(n))
        S = a.sum()
        # offsets inside the case-(3) window [n2, min(n1+n2, n3)] and below / above it
        for frac in (-3.0, 0.1, 0.5, 0.9, 4.0):
            d = a[1] + frac * a[0]
            d0 = d - 0.5 * S
            t = F(d0) + (F(a[0]) + F(a[1]) + F(a[2])) / 2
            tot = F(0)
            for v in itertools.product((0, 1), repeat=3):
                r = t - sum(F(ai) for ai, vi in zip(a, v) if vi)
                if r > 0:
                    tot += (-1) ** sum(v) * r ** 3
            exact = float(tot / (6 * F(a[0]) * F(a[1]) * F(a[2])))
            got = float(oracle.volume(d0, *n))
            model = 1e-15 + 1e-15 * d ** 3 / (6 * a[0] * a[1] * a[2])
            worst_v = max(worst_v, abs(got - exact) / model)
            back = float(oracle.solve(exact, *n))
            worst_d = max(worst_d, abs(back - d0))
    assert worst_v < 1.0 and worst_d < 1e-8, (worst_v, worst_d)


def test_fp32_inputs_are_promoted_exactly():
    n = unit(RNG.standard_normal((1000, 3))).astype(np.float32)
    V0 = RNG.random(1000).astype(np.float32)
    a = oracle.solve(V0, n[:, 0], n[:, 1], n[:, 2])
    b = oracle.solve(V0.astype(np.float64), *(n[:, i].astype(np.float64) for i in range(3)))
    assert a.dtype == np.float64 and np.array_equal(a, b)


def test_degenerate_inputs():
    assert oracle.solve(0.3, 0.0, 0.0, 0.0) == 0.0                       # reading R6
    assert oracle.volume(0.0, 0.0, 0.0, 0.0) == 0.5
    assert math.isnan(float(oracle.solve(float("nan"), 1.0, 0.0, 0.0)))
    # tiny but non-zero smallest component: no division blow-up anywhere on [0,1]
    for eps in (1e-3, 1e-8, 1e-20, 1e-38):
        n = unit([eps, 0.6, 0.8])
        V0 = np.linspace(0, 1, 1001)
        d = oracle.solve(V0, *n)
        assert np.all(np.isfinite(d)) and np.all(np.diff(d) >= 0)
        n2d = unit([0.0, 0.6, 0.8])
        assert np.max(np.abs(d - oracle.solve(V0, *n2d))) < 2 * eps + 1e-12


# ----------------------------------------------------------------------------------
# worked examples
# ----------------------------------------------------------------------------------
def _golden_rows():
    rows = []
    env = {"sqrt": math.sqrt, "__builtins__": {}}
    with open(os.path.join(HERE, "golden", "worked_examples.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            a, V0, d0, why = [s.strip() for s in line.split("|", 3)]
            a = [float(x) for x in a.split()]
            rows.append((a, float(eval(V0, env)), float(eval(d0, env)), why))
    return rows


@pytest.mark.parametrize("a,V0,d0,why", _golden_rows())
def test_p13_worked_examples(a, V0, d0, why):
    a = np.asarray(a)
    for perm in itertools.permutations(range(3)):
        for sg in itertools.product((1.0, -1.0), repeat=3):
            # mirroring a component reflects the cube onto itself: same V0 <-> d0 map
            n = unit(a[list(perm)] * np.asarray(sg))
            assert abs(float(oracle.solve(V0, *n)) - d0) < 1e-12, why
            assert abs(float(oracle.solve(1.0 - V0, *n)) + d0) < 1e-12, why
            assert abs(float(oracle.volume(d0, *n)) - V0) < 1e-12, why
