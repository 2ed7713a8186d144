"""fp64 CPU oracle for the plane-sphere problem of sect. 3 -- TEST INFRASTRUCTURE, NOT PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s oracle legs may import this
module; it shares no code with the CUDA path.  PAPER.md = /root/reference/PAPER.md.

What it computes: a sphere of unit volume, radius r = (3/(4 pi))^(1/3)
(eq. (34)), centred at the origin, is cut by the plane n.x = d0; only the offset matters, not
the direction.

    sphere_volume(d0)  eq. (37), the spherical-cap formula, written out as printed:
                       V0 = pi/3 (r + d0)^2 (2r - d0),  d0 clamped to [-r, r]
    sphere_solve(V0)   the unique d0 in [-r, r] with sphere_volume(d0) = V0 (eq. (36)): the
                       plain definition, by bisection of eq. (37) down to an interval narrower
                       than 1e-15.  It does NOT use the paper's closed form eq. (38); that
                       formula is one of the pins (tests/test_sphere_pins.py).

Readings: V0 <= 0 -> -r, V0 >= 1 -> +r (ends of the interval, as for the cube); numpy fp64
throughout; inputs are the fp32 values the CUDA path sees, promoted exactly.

Pins (tests/test_sphere_pins.py): eq. (38) as printed; the end points and the centre; the
symmetry d0(1 - V0) = -d0(V0); dV0/dd0 = area of the cut disc pi (r^2 - d0^2); the cap of
height r/2 has volume 5/32 exactly; Monte-Carlo counting of points in the ball.
"""
from __future__ import annotations

import numpy as np

R = (3.0 / (4.0 * np.pi)) ** (1.0 / 3.0)          # eq. (34)


def sphere_volume(d0) -> np.ndarray:
    """eq. (37)."""
    d = np.clip(np.asarray(d0, dtype=np.float64), -R, R)
    return np.pi / 3.0 * (R + d) ** 2 * (2.0 * R - d)


def sphere_solve(V0) -> np.ndarray:
    """Bisection of eq. (37) on [-r, r] (eq. (36))."""
    v = np.asarray(V0, dtype=np.float64)
    lo = np.full(v.shape, -R)
    hi = np.full(v.shape, R)
    for _ in range(64):
        mid = 0.5 * (lo + hi)
        below = sphere_volume(mid) < v
        lo = np.where(below, mid, lo)
        hi = np.where(below, hi, mid)
    out = 0.5 * (lo + hi)
    out = np.where(v <= 0.0, -R, out)
    out = np.where(v >= 1.0, R, out)
    return out
