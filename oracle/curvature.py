"""fp64 CPU oracle for the curvature calculation of sect. 4 / appendix B -- TEST INFRASTRUCTURE,
NOT PRODUCT.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s oracle legs may
import this module; it shares no code with the CUDA path.  PAPER.md = /root/reference/PAPER.md.

What it computes (eq. (41)): for an interface lattice point, from the 3^3
neighbourhood of fill levels phi_0..phi_26, the mean curvature kappa of the interface.  It
follows the paper's algorithm step by step, in the paper's order and notation, vectorised
over cells only (numpy fp64; the PLIC offsets come from the bisection oracle ``oracle.solve``):

  1. n = n_PY, the Parker-Youngs normal, eq. (54) with the weights of eq. (55) (4, 2, 1 for
     |e_i| = 1, sqrt2, sqrt3), e_i the 27 directions of eq. (53)
  2. b_z = n, b_y = (b_z x r)/|b_z x r|, b_x = b_y x b_z with the fixed vector r of eq. (42)
                                                                          PAPER.md:351-361
  3. for every neighbour i = 1..26 with 0 < phi_i < 1 (interface points only):
     p_i = (e_i.b_x, e_i.b_y, e_i.b_z + d0(phi_i, n) - d0(phi_0, n))       eq. (46)
  4. M = sum Q_i Q_i^T, b = sum z_i Q_i with Q = (x^2, y^2, xy, x, y)       eq. (47)-(49), (69)
  5. M x = b, x = (A, B, C, H, I)                                          eq. (70)
     (``numpy.linalg.solve`` serves as the LU decomposition).  With k < 5 points the number of
     fitting parameters is reduced to k: the leading k x k block is solved and the remaining
     parameters stay zero.
  6. kappa = (A (I^2+1) + B (H^2+1) - C H I) / (H^2 + I^2 + 1)^(3/2)        eq. (63)

Readings (each also in DESIGN.md):
  C1  Sign.  eq. (54) makes n point out of the fluid; z is the height along n; a convex fluid
      body (drop) then has A, B < 0 and eq. (63) gives kappa = -1/R, whereas the text speaks
      of kappa = 1/R for drops.  The oracle returns eq. (63) literally;
      tests compare -kappa with 1/R.
  C2  Cells that are not interface (phi_0 <= 0 or >= 1), cells on the lattice border (no full
      3^3 neighbourhood), a vanishing gradient sum in eq. (54), and cells without any interface
      neighbour get kappa = 0 (the paper is silent).
  C3  "Reducing dimensionality" keeps the first k of (A, B, C, H, I).
  C4  A singular (k x k) system is outside the comparison (the paper's LU has no pivot check);
      the oracle reports NaN for it and the parity tests exclude such cells.
  C5  Lattice layout: phi[z, y, x] (x fastest), cell spacing 1, e_i = (dx, dy, dz).

Pins (tests/test_curvature_pins.py): eq. (63) against the mean curvature of a sphere graph at
an off-pole point; exact recovery of a known paraboloid by the least-squares fit, also with
k < 5 points; the PY normal of a linear field; kappa = 0 for planar interfaces whose PY normal
is exact; -kappa R -> 1 on sphere lattices and -kappa R -> 1/2 on cylinders; invariance under
the choice of r and under lattice mirrors.
"""
from __future__ import annotations

import numpy as np

import oracle as _plic_oracle

R_VEC = np.array([0.56270900, 0.32704452, 0.75921047])           # eq. (42)

# e_i, i = 0..26 (eq. (53)): index = (dx+1) + 3 (dy+1) + 9 (dz+1); e_13 is the centre
E = np.array([(dx, dy, dz) for dz in (-1, 0, 1) for dy in (-1, 0, 1) for dx in (-1, 0, 1)],
             dtype=np.float64)
CENTRE = 13
_W = np.array([0.0, 4.0, 2.0, 1.0])[np.abs(E).sum(axis=1).astype(int)]   # eq. (55)


def py_normal(phi27: np.ndarray) -> np.ndarray:
    """eq. (54): n_PY = -sum w_i e_i phi_i / |.|; zero rows where the sum vanishes (C2)."""
    g = (phi27[:, :, None] * (_W[:, None] * E)[None, :, :]).sum(axis=1)
    norm = np.sqrt((g * g).sum(axis=1))
    n = np.zeros_like(g)
    ok = norm > 0.0
    n[ok] = -g[ok] / norm[ok, None]
    return n


def basis(n: np.ndarray, r=R_VEC):
    """eq. (43)-(45)."""
    bz = n
    by = np.cross(bz, np.asarray(r, dtype=np.float64)[None, :])
    by = by / np.sqrt((by * by).sum(axis=1))[:, None]
    bx = np.cross(by, bz)
    return bx, by, bz


def curvature_from_fit(x5: np.ndarray) -> np.ndarray:
    """eq. (63)."""
    A, B, C, H, I = (x5[:, j] for j in range(5))
    return (A * (I * I + 1.0) + B * (H * H + 1.0) - C * H * I) / np.sqrt(H * H + I * I + 1.0) ** 3


def paraboloid_fit(x, y, z, use) -> np.ndarray:
    """Steps 4 and 5 for a batch: x, y, z, use are [m, 26]; returns (A, B, C, H, I) per row."""
    m = x.shape[0]
    Q = np.stack([x * x, y * y, x * y, x, y], axis=2) * use[:, :, None]            # eq. (49)
    M = np.einsum("mia,mib->mab", Q, Q)                                            # eq. (69)
    b = np.einsum("mia,mi->ma", Q, z * use)
    count = use.sum(axis=1).astype(int)
    out = np.zeros((m, 5))
    for k in range(1, 6):
        rows = np.where(count == k)[0] if k < 5 else np.where(count >= 5)[0]
        for j in rows:
            try:
                out[j, :k] = np.linalg.solve(M[j, :k, :k], b[j, :k])               # eq. (70)
            except np.linalg.LinAlgError:
                out[j, :] = np.nan                                                 # C4
    return out


def curvature_cells(phi27: np.ndarray, r=R_VEC) -> np.ndarray:
    """kappa for cells given as rows of 27 fill levels (ordering of E); the centre must be an
    interface point.  Returns [m] fp64."""
    phi27 = np.asarray(phi27, dtype=np.float64)
    m = phi27.shape[0]
    n = py_normal(phi27)                                                           # step 1
    good = (n * n).sum(axis=1) > 0.0
    kappa = np.zeros(m)
    if not good.any():
        return kappa
    p = phi27[good]
    nn = n[good]
    bx, by, bz = basis(nn, r)                                                      # step 2
    nb = np.array([i for i in range(27) if i != CENTRE])
    phi_nb = p[:, nb]
    use = ((phi_nb > 0.0) & (phi_nb < 1.0)).astype(np.float64)                     # step 3
    rep = lambda a: np.repeat(a[:, None], 26, axis=1)
    d_nb = _plic_oracle.solve(phi_nb, rep(nn[:, 0]), rep(nn[:, 1]), rep(nn[:, 2]))
    d_0 = _plic_oracle.solve(p[:, CENTRE], nn[:, 0], nn[:, 1], nn[:, 2])
    e = E[nb]
    x = bx @ e.T
    y = by @ e.T
    z = bz @ e.T + d_nb - d_0[:, None]                                             # eq. (46)
    fit = paraboloid_fit(x, y, z, use)                                             # steps 4, 5
    k = curvature_from_fit(fit)                                                    # step 6
    k = np.where(use.sum(axis=1) > 0, k, 0.0)
    kappa[good] = k
    return kappa


def fit_diagnostics(phi27: np.ndarray, r=R_VEC):
    """Test diagnostics, not part of the method: per cell the number of interface neighbours, the
    2-norm condition number of the k x k system of eq. (70) (inf where there is none) and its
    smallest eigenvalue (0 where there is none)."""
    phi27 = np.asarray(phi27, dtype=np.float64)
    n = py_normal(phi27)
    nb = np.array([i for i in range(27) if i != CENTRE])
    use = ((phi27[:, nb] > 0.0) & (phi27[:, nb] < 1.0)).astype(np.float64)
    count = use.sum(axis=1).astype(int)
    cond = np.full(phi27.shape[0], np.inf)
    lam_min = np.zeros(phi27.shape[0])
    good = ((n * n).sum(axis=1) > 0.0) & (count > 0)
    if good.any():
        bx, by, _ = basis(n[good], r)
        e = E[nb]
        x, y = bx @ e.T, by @ e.T
        Q = np.stack([x * x, y * y, x * y, x, y], axis=2) * use[good][:, :, None]
        M = np.einsum("mia,mib->mab", Q, Q)
        c = np.empty(M.shape[0])
        lm = np.empty(M.shape[0])
        for j, k in enumerate(np.minimum(count[good], 5)):
            ev = np.linalg.eigvalsh(M[j, :k, :k])
            lm[j] = max(ev[0], 0.0)
            c[j] = ev[-1] / ev[0] if ev[0] > 0.0 else np.inf
        cond[good] = c
        lam_min[good] = lm
    return count, cond, lam_min


def gather27(phi: np.ndarray, idx: np.ndarray) -> np.ndarray:
    """The 3^3 neighbourhoods (ordering of E) of the interior cells idx = [m, 3] as (z, y, x)."""
    out = np.empty((idx.shape[0], 27))
    for i, (dx, dy, dz) in enumerate(E.astype(int)):
        out[:, i] = phi[idx[:, 0] + dz, idx[:, 1] + dy, idx[:, 2] + dx]
    return out


def curvature_lattice(phi: np.ndarray, r=R_VEC) -> np.ndarray:
    """kappa on the whole lattice phi[z, y, x]; 0 where C2 says so."""
    phi = np.asarray(phi, dtype=np.float64)
    kappa = np.zeros(phi.shape)
    inner = np.zeros(phi.shape, dtype=bool)
    inner[1:-1, 1:-1, 1:-1] = True
    idx = np.argwhere((phi > 0.0) & (phi < 1.0) & inner)
    if len(idx):
        kappa[idx[:, 0], idx[:, 1], idx[:, 2]] = curvature_cells(gather27(phi, idx), r)
    return kappa
