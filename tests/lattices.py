"""Fill-level lattices for the curvature tests.  phi of a cell is the volume the half-space
tangent to the body at the point nearest to the cell centre cuts out of the cell -- the
paper's own initialisation "with the inverse PLIC algorithm" -- evaluated with
the oracle's forward map, which is why this lives in tests/ and not in gen/.
Layout phi[z, y, x], cell (i, j, k) centred at (i + 1/2, j + 1/2, k + 1/2)."""
import numpy as np

import oracle


def _centres(shape):
    nz, ny, nx = shape
    z, y, x = np.meshgrid(np.arange(nz) + 0.5, np.arange(ny) + 0.5, np.arange(nx) + 0.5, indexing="ij")
    return x, y, z


def _from_signed_distance(sd, nx_, ny_, nz_):
    """sd = signed distance of the cell centre to the surface along the outward normal n (> 0 outside
    the fluid).  The plane n.(x - c) = -sd bounds the fluid, so phi = V0(d0 = -sd, n)."""
    phi = np.where(sd > 0, 0.0, 1.0)
    near = np.abs(sd) < 1.0
    phi[near] = oracle.volume(-sd[near], nx_[near], ny_[near], nz_[near])
    return phi.astype(np.float32)


def sphere(shape, centre, R):
    x, y, z = _centres(shape)
    dx, dy, dz = x - centre[0], y - centre[1], z - centre[2]
    r = np.sqrt(dx * dx + dy * dy + dz * dz)
    r = np.maximum(r, 1e-300)
    return _from_signed_distance(r - R, dx / r, dy / r, dz / r)


def cylinder(shape, centre_xy, R):
    """Axis along z."""
    x, y, z = _centres(shape)
    dx, dy = x - centre_xy[0], y - centre_xy[1]
    r = np.maximum(np.sqrt(dx * dx + dy * dy), 1e-300)
    return _from_signed_distance(r - R, dx / r, dy / r, np.zeros_like(r))


def plane(shape, normal, offset):
    """Fluid where normal.x <= offset."""
    n = np.asarray(normal, dtype=np.float64)
    n = n / np.sqrt((n * n).sum())
    x, y, z = _centres(shape)
    sd = n[0] * x + n[1] * y + n[2] * z - offset
    o = np.ones_like(sd)
    return _from_signed_distance(sd, n[0] * o, n[1] * o, n[2] * o)
