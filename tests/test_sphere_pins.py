"""Pins of the plane-sphere oracle (oracle/sphere.py) against what the paper and geometry fix
(sect. 3).  CPU only."""
import numpy as np

from oracle import sphere

R = (3.0 / (4.0 * np.pi)) ** (1.0 / 3.0)


def test_radius_gives_unit_volume():
    # eq. (34): 1 = 4/3 pi r^3
    assert abs(4.0 / 3.0 * np.pi * sphere.R ** 3 - 1.0) < 1e-15
    assert abs(sphere.R - R) < 1e-16


def test_end_points_centre_and_range():
    assert sphere.sphere_volume(-R) == 0.0
    assert abs(sphere.sphere_volume(R) - 1.0) < 1e-15
    assert abs(sphere.sphere_volume(0.0) - 0.5) < 1e-15
    assert sphere.sphere_solve(0.0) == -R and sphere.sphere_solve(1.0) == R
    assert abs(sphere.sphere_solve(0.5)) < 1e-15
    # outside the domain: clamped (readings in the oracle's header)
    assert sphere.sphere_solve(-0.25) == -R and sphere.sphere_solve(1.5) == R
    assert sphere.sphere_volume(2.0) == sphere.sphere_volume(R)


def test_cap_of_half_radius_is_5_32():
    # textbook cap of height h: pi h^2 (3r - h)/3; h = r/2 -> 5 pi r^3 / 24 = 5/32 with eq. (34)
    assert abs(sphere.sphere_volume(-R / 2) - 5.0 / 32.0) < 1e-15
    assert abs(sphere.sphere_solve(5.0 / 32.0) + R / 2) < 1e-14
    assert abs(sphere.sphere_solve(27.0 / 32.0) - R / 2) < 1e-14


def _golden_rows():
    import os
    rows = []
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "sphere_examples.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                v, d, why = [x.strip() for x in line.split("|", 2)]
                rows.append((eval(v), eval(d), why))
    return rows


def test_golden_caps():
    rows = _golden_rows()
    assert len(rows) >= 7
    for V0, d_over_r, why in rows:
        ok = abs(sphere.sphere_solve(V0) - d_over_r * R) < 1e-13 and abs(sphere.sphere_volume(d_over_r * R) - V0) < 1e-14
        # the row marked "negative control" states a wrong volume on purpose: the oracle must reject it
        assert ok != ("negative control" in why), (V0, d_over_r, why)


def test_closed_form_eq38():
    # eq. (38) exactly as printed, against the bisection
    V = np.concatenate([np.linspace(0.0, 1.0, 4001), 10.0 ** np.linspace(-12, -1, 200),
                        1.0 - 10.0 ** np.linspace(-12, -1, 200)])
    d38 = np.cbrt(6.0 / np.pi) * np.sin(np.pi / 6.0 - np.arctan2(2.0 * np.sqrt(np.maximum(V - V * V, 0.0)),
                                                                 2.0 * V - 1.0) / 3.0)
    d = sphere.sphere_solve(V)
    # eq. (38) evaluated in fp64 loses digits of V near 1 (2V - 1), hence 1e-9 there
    assert np.max(np.abs(d - d38)) < 1e-9
    mid = (V > 1e-3) & (V < 1 - 1e-3)
    assert np.max(np.abs(d[mid] - d38[mid])) < 1e-13


def test_symmetry_monotone_round_trip():
    rng = np.random.default_rng(3)
    V = rng.random(20000)
    d = sphere.sphere_solve(V)
    assert np.max(np.abs(sphere.sphere_solve(1.0 - V) + d)) < 1e-13
    assert np.max(np.abs(sphere.sphere_volume(d) - V)) < 1e-14
    s = np.sort(V)
    assert np.all(np.diff(sphere.sphere_solve(s)) >= 0.0)
    dd = np.linspace(-R, R, 5001)
    assert np.all(np.diff(sphere.sphere_volume(dd)) > 0.0)
    assert np.max(np.abs(sphere.sphere_volume(-dd) - (1.0 - sphere.sphere_volume(dd)))) < 1e-15


def test_derivative_is_disc_area():
    d = np.linspace(-0.9 * R, 0.9 * R, 101)
    h = 1e-6
    num = (sphere.sphere_volume(d + h) - sphere.sphere_volume(d - h)) / (2 * h)
    assert np.max(np.abs(num - np.pi * (R * R - d * d))) < 1e-8


def test_monte_carlo_ball():
    rng = np.random.default_rng(5)
    p = (rng.random((400000, 3)) * 2 - 1) * R
    inside = (p ** 2).sum(axis=1) <= R * R
    for d0 in (-0.4, -0.1, 0.0, 0.25, 0.5):
        # any direction: use z
        frac = np.count_nonzero(inside & (p[:, 2] <= d0)) / np.count_nonzero(inside)
        assert abs(frac - sphere.sphere_volume(d0)) < 4e-3
