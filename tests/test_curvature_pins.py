"""Pins of the curvature oracle (oracle/curvature.py) against what the paper and geometry fix
(sect. 4, appendix B).  CPU only."""
import os
import sys

import numpy as np

from oracle import curvature as oc

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import lattices  # noqa: E402


def test_directions_and_weights():
    # eq. (53): the 27 vectors of {-1,0,1}^3; eq. (55): 6 x 4, 12 x 2, 8 x 1, centre 0
    assert len({tuple(e) for e in oc.E}) == 27 and np.all(np.abs(oc.E) <= 1)
    assert tuple(oc.E[oc.CENTRE]) == (0, 0, 0)
    w = oc._W
    l2 = (oc.E ** 2).sum(axis=1)
    assert np.all(w[l2 == 1] == 4) and np.all(w[l2 == 2] == 2) and np.all(w[l2 == 3] == 1) and w[oc.CENTRE] == 0
    assert (l2 == 1).sum() == 6 and (l2 == 2).sum() == 12 and (l2 == 3).sum() == 8
    # sum_i w_i e_i e_i^T = 32 I (eq. (51) has 18 I for unit weights)
    assert np.allclose(np.einsum("i,ia,ib->ab", w, oc.E, oc.E), 32 * np.eye(3))


def test_py_normal_of_linear_field():
    # phi_i = c + g.e_i  ->  sum w_i e_i phi_i = 32 g  ->  n = -g/|g| exactly (eq. (54))
    rng = np.random.default_rng(1)
    g = rng.standard_normal((200, 3)) * 0.1
    phi = 0.5 + g @ oc.E.T
    n = oc.py_normal(phi)
    assert np.max(np.abs(n + g / np.linalg.norm(g, axis=1)[:, None])) < 1e-13
    assert np.all(oc.py_normal(np.full((3, 27), 0.5)) == 0.0)          # C2: vanishing gradient


def test_basis_is_orthonormal_right_handed():
    rng = np.random.default_rng(2)
    n = rng.standard_normal((100, 3))
    n /= np.linalg.norm(n, axis=1)[:, None]
    bx, by, bz = oc.basis(n)
    for a in (bx, by, bz):
        assert np.max(np.abs(np.linalg.norm(a, axis=1) - 1)) < 1e-13
    assert np.max(np.abs((bx * by).sum(1))) < 1e-13 and np.max(np.abs((bx * bz).sum(1))) < 1e-13
    assert np.max(np.abs(np.cross(bx, by) - bz)) < 1e-13               # b_x x b_y = b_z
    assert np.all(bz == n)
    assert np.max(np.abs((by * oc.R_VEC).sum(1))) < 1e-13              # b_y is normal to r (eq. (44))


def test_eq63_is_the_mean_curvature_of_a_sphere_graph():
    # z = f(x,y) = -sqrt(R^2 - (x-x0)^2 - (y-y0)^2): the lower half of a sphere seen from inside
    # has mean curvature +1/R at every point, the upper half (-f) has -1/R.  The paraboloid
    # with the same derivatives at the origin, A = fxx/2, B = fyy/2, C = fxy, H = fx, I = fy
    # (eq. (58)-(62)), must reproduce it through eq. (63).
    rng = np.random.default_rng(3)
    for _ in range(50):
        R = rng.uniform(2, 50)
        x0, y0 = rng.uniform(-0.6, 0.6, 2) * R
        s = np.sqrt(R * R - x0 * x0 - y0 * y0)
        fx, fy = -x0 / s, -y0 / s                       # derivatives of f at (0, 0)
        fxx = 1 / s + x0 * x0 / s ** 3
        fyy = 1 / s + y0 * y0 / s ** 3
        fxy = x0 * y0 / s ** 3
        x5 = np.array([[fxx / 2, fyy / 2, fxy, fx, fy]])
        assert abs(oc.curvature_from_fit(x5)[0] - 1 / R) < 1e-12 / R
        assert abs(oc.curvature_from_fit(-x5)[0] + 1 / R) < 1e-12 / R
    # saddle z = x^2 - y^2: mean curvature 0; cylinder z = x^2/(2R): 1/(2R)
    assert oc.curvature_from_fit(np.array([[1.0, -1.0, 0, 0, 0]]))[0] == 0.0
    assert abs(oc.curvature_from_fit(np.array([[0.05, 0.0, 0, 0, 0]]))[0] - 0.05) < 1e-15


def test_least_squares_recovers_a_paraboloid():
    rng = np.random.default_rng(4)
    for k in (5, 8, 26):
        co = rng.standard_normal((20, 5))
        x = rng.uniform(-1.5, 1.5, (20, 26))
        y = rng.uniform(-1.5, 1.5, (20, 26))
        use = np.zeros((20, 26))
        use[:, :k] = 1
        z = co[:, 0:1] * x * x + co[:, 1:2] * y * y + co[:, 2:3] * x * y + co[:, 3:4] * x + co[:, 4:5] * y
        z = z + 100.0 * (1 - use)                                    # unused points must not matter
        fit = oc.paraboloid_fit(x, y, z, use)
        assert np.max(np.abs(fit - co)) < 1e-6          # normal equations: cond(M) = cond(Q)^2
    # fewer than five points: the first k parameters only
    for k in (1, 2, 3, 4):
        co = np.zeros((10, 5))
        co[:, :k] = rng.standard_normal((10, k))
        x = rng.uniform(0.5, 1.5, (10, 26))
        y = rng.uniform(0.5, 1.5, (10, 26))
        use = np.zeros((10, 26))
        use[:, 3:3 + k] = 1
        z = co[:, 0:1] * x * x + co[:, 1:2] * y * y + co[:, 2:3] * x * y + co[:, 3:4] * x + co[:, 4:5] * y
        fit = oc.paraboloid_fit(x, y, z, use)
        assert np.max(np.abs(fit - co)) < 1e-6 and np.all(fit[:, k:] == 0.0)


def test_planar_interfaces_have_zero_curvature():
    # planes whose Parker-Youngs normal is exact by symmetry: the PLIC points are then coplanar
    for normal, off in (((1, 0, 0), 7.3), ((0, 0, -1), -6.6), ((1, 1, 0), 14.2), ((1, -1, 1), 5.1)):
        phi = lattices.plane((14, 14, 14), normal, off)
        k = oc.curvature_lattice(phi)
        inner = (phi[1:-1, 1:-1, 1:-1] > 0) & (phi[1:-1, 1:-1, 1:-1] < 1)
        assert inner.sum() > 50
        assert np.max(np.abs(k)) < 1e-6, (normal, np.max(np.abs(k)))   # phi is stored in fp32
    # a general plane: the PY normal is only approximate, kappa stays small
    phi = lattices.plane((16, 16, 16), (0.3, 0.5, 0.81), 12.9)
    assert np.max(np.abs(oc.curvature_lattice(phi))) < 0.05


def test_sphere_and_cylinder():
    # C1: eq. (63) with the outward normal of eq. (54) gives -1/R for a drop
    for R, L in ((8, 24), (12, 32), (20, 48)):
        phi = lattices.sphere((L, L, L), (L / 2 + 0.3, L / 2 - 0.3, L / 2 + 0.1), R)
        k = oc.curvature_lattice(phi)
        kk = -k[k != 0] * R
        assert len(kk) > 1000 and not np.isnan(kk).any()
        assert abs(kk.mean() - 1.0) < 0.02                               # mean within 2 %
        assert np.abs(kk - 1.0).mean() < 0.08                            # eq. (50) L1 error
    # bubble: fluid outside, curvature +1/R
    phi = 1.0 - lattices.sphere((32, 32, 32), (16.2, 15.9, 16.4), 12)
    k = oc.curvature_lattice(phi.astype(np.float32))
    assert abs(k[k != 0].mean() * 12 - 1.0) < 0.02
    # cylinder: mean curvature 1/(2R)
    phi = lattices.cylinder((12, 40, 40), (20.3, 19.8), 14)
    k = oc.curvature_lattice(phi)
    kk = -k[k != 0] * 14
    assert abs(kk.mean() - 0.5) < 0.02


def test_invariance_under_r_and_mirrors():
    phi = lattices.sphere((26, 26, 26), (13.2, 12.7, 13.1), 9)
    k0 = oc.curvature_lattice(phi)
    # the five-parameter fit is invariant under rotations of (b_x, b_y) about b_z, i.e. under r
    k1 = oc.curvature_lattice(phi, r=(0.1, -0.7, 0.2))
    full = k0 != 0
    assert np.max(np.abs(k0[full] - k1[full])) < 1e-7
    # mirrored lattice -> mirrored curvature field
    k2 = oc.curvature_lattice(phi[:, :, ::-1].copy())[:, :, ::-1]
    k3 = oc.curvature_lattice(phi.transpose(2, 1, 0).copy()).transpose(2, 1, 0)
    assert np.max(np.abs(k0 - k2)) < 1e-7 and np.max(np.abs(k0 - k3)) < 1e-7


def test_non_interface_and_border_cells_are_zero():
    phi = lattices.sphere((16, 16, 16), (8, 8, 2.0), 6)                   # cut by the z = 0 border
    k = oc.curvature_lattice(phi)
    assert np.all(k[0] == 0) and np.all(k[:, 0] == 0) and np.all(k[:, :, -1] == 0)
    assert np.all(k[(phi <= 0) | (phi >= 1)] == 0)
