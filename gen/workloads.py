"""Seeded fp32 SoA workload generators for the PLIC path.  See gen/__init__.py.

Nothing here evaluates the PLIC forward or inverse map, classifies an
intersection case, or sorts a normal: the generators only draw normals and
volumes with the distributions BASELINE.json's configs name.  (The
case-stratified configs[2] needs the oracle's forward map and classifier and
therefore lives in oracle/stratified.c / oracle/stratified.py, not here.)
"""
from __future__ import annotations

from concurrent.futures import ThreadPoolExecutor
import os

import numpy as np

CHUNK = 1 << 20          # cells per Philox chunk; part of the recipe, do not change

# stream ids (second Philox key word): one per workload family
_STREAM_SPHERE = 1
_STREAM_EDGE = 2
_STREAM_SNAP = 3
_STREAM_PAPER = 4
_STREAM_PAPER_NORMALS = 5

_INV_SQRT2_F32 = np.float32(0.70710677)


def _rng(seed: int, stream: int, chunk: int) -> np.random.Generator:
    key = np.array([seed, stream], dtype=np.uint64)
    counter = np.array([0, 0, 0, chunk], dtype=np.uint64)
    return np.random.Generator(np.random.Philox(key=key, counter=counter))


def _unit_rows(g: np.ndarray) -> np.ndarray:
    """Normalise the rows of g (fp64) to L2 length 1; a zero row becomes (0,0,1)."""
    r = np.sqrt(np.einsum("ij,ij->i", g, g))
    bad = r == 0.0
    if bad.any():
        g = g.copy()
        g[bad] = (0.0, 0.0, 1.0)
        r[bad] = 1.0
    return g / r[:, None]


def _chunk_spans(start: int, count: int):
    """(chunk index, lo, hi, out offset) for the cells [start, start+count)."""
    out = 0
    c = start // CHUNK
    while out < count:
        lo = (start + out) - c * CHUNK
        hi = min(CHUNK, lo + (count - out))
        yield c, lo, hi, out
        out += hi - lo
        c += 1


def _run_chunks(fn, start, count, workers, dtype=np.float32):
    V0 = np.empty(count, dtype=dtype)
    nx = np.empty(count, dtype=dtype)
    ny = np.empty(count, dtype=dtype)
    nz = np.empty(count, dtype=dtype)

    def work(span):
        c, lo, hi, o = span
        v, n = fn(c)
        m = hi - lo
        V0[o:o + m] = v[lo:hi]
        nx[o:o + m] = n[lo:hi, 0]
        ny[o:o + m] = n[lo:hi, 1]
        nz[o:o + m] = n[lo:hi, 2]

    spans = list(_chunk_spans(start, count))
    if workers is None:
        workers = min(len(spans), os.cpu_count() or 1, 16)
    if workers <= 1 or len(spans) <= 1:
        for s in spans:
            work(s)
    else:
        with ThreadPoolExecutor(max_workers=workers) as ex:
            list(ex.map(work, spans))
    return V0, nx, ny, nz


def random_sphere(N: int, seed: int, start: int = 0, workers: int | None = None, dtype=np.float32):
    """Config 1 (random part) and config 2: normals uniform on the unit sphere
    (normalised i.i.d. N(0,1) 3-vectors), V0 ~ U[0,1).  Returns (V0, nx, ny, nz)
    for the cells [start, start+N) of the stream keyed by `seed`, in `dtype`: fp32 (the
    paper's type), or the same fp64 draws rounded once to fp16 or kept in fp64 (the
    storage variants plic_solve_h / plic_solve_f64)."""
    def chunk(c):
        rng = _rng(seed, _STREAM_SPHERE, c)
        g = rng.standard_normal((CHUNK, 3))
        u = rng.random(CHUNK)
        return u.astype(dtype), _unit_rows(g).astype(dtype)
    return _run_chunks(chunk, start, N, workers, dtype)


EDGE_V0 = np.array([0.0, 0.5, 1.0, 1e-7, 1.0 - 1e-7], dtype=np.float32)


def edge_cells(count: int = 4096, seed: int = 0, dtype=np.float32):
    """Config 1 edge part: normals with one or two components exactly 0 (random
    signs, survivors random and renormalised; a single survivor is exactly +-1),
    V0 cycling through {0, 0.5, 1, 1e-7, 1-1e-7} (the last rounds to 0.99999988f).
    Cell j: V0 = EDGE_V0[j % 5]; (j // 5) % 2 == 0 -> one zero component, else two."""
    rng = _rng(seed, _STREAM_EDGE, 0)
    g = rng.standard_normal((count, 3))
    k = rng.integers(0, 3, size=count)            # which component is zeroed / survives
    j = np.arange(count)
    two = ((j // 5) % 2) == 1
    keep = np.ones((count, 3), dtype=bool)
    keep[~two, k[~two]] = False                   # one zero: drop component k
    keep[two] = False
    keep[two, k[two]] = True                      # two zeros: only component k survives
    g = np.where(keep, g, 0.0)
    n = _unit_rows(g).astype(dtype)
    # the five volumes in `dtype`: 1e-7 is subnormal in fp16 (1.19e-7) and 1 - 1e-7 rounds to 1 there
    V0 = np.array([0.0, 0.5, 1.0, 1e-7, 1.0 - 1e-7], dtype=np.float64).astype(dtype)[j % 5].copy()
    return V0, n[:, 0].copy(), n[:, 1].copy(), n[:, 2].copy()


def config1(seed: int = 0, n_random: int = 1 << 20, n_edge: int = 4096, dtype=np.float32):
    """BASELINE.json configs[0]: n_random random cells followed by n_edge edge cells."""
    a = random_sphere(n_random, seed, dtype=dtype)
    b = edge_cells(n_edge, seed, dtype=dtype)
    return tuple(np.concatenate([x, y]) for x, y in zip(a, b))


def snapped_beta(N: int, seed: int, start: int = 0, workers: int | None = None):
    """Config 4: with probability 1/2 the normal is snapped -- half of those to a
    signed coordinate axis, half to a signed face diagonal (two components
    +-0.70710677f, one exactly 0) -- else uniform on the sphere;
    V0 ~ Beta(1/2, 1/2) via V0 = sin^2(pi U / 2)."""
    def chunk(c):
        rng = _rng(seed, _STREAM_SNAP, c)
        g = rng.standard_normal((CHUNK, 3))
        u = rng.random(CHUNK)
        sel = rng.random(CHUNK)
        k = rng.integers(0, 3, size=CHUNK)
        n = _unit_rows(g).astype(np.float32)
        sgn = np.where(g < 0.0, np.float32(-1.0), np.float32(1.0)).astype(np.float32)
        idx = np.arange(CHUNK)
        axis = sel < 0.25
        diag = (sel >= 0.25) & (sel < 0.5)
        onehot = np.zeros((CHUNK, 3), dtype=bool)
        onehot[idx, k] = True
        n = np.where(axis[:, None], np.where(onehot, sgn, np.float32(0.0)), n)
        n = np.where(diag[:, None], np.where(onehot, np.float32(0.0), sgn * _INV_SQRT2_F32), n)
        v = np.sin(0.5 * np.pi * u) ** 2
        return v.astype(np.float32), n.astype(np.float32)
    return _run_chunks(chunk, start, N, workers)


def paper_benchmark_set(n_normals: int, L: int, seed: int):
    """The paper's own benchmark shape: normal 0 is (1,0,0),
    normal 1 is (1/sqrt2, 1/sqrt2, 0), the next n_normals/8 - 2 are random 2D
    directions in the x-y plane, the rest random 3D directions; for each normal V0
    takes L equally spaced values in [0,1] including both ends.  Returns the
    n_normals*L cells, normal-major."""
    rng = _rng(seed, _STREAM_PAPER, 0)
    g = rng.standard_normal((n_normals, 3))
    n2d = max(n_normals // 8, 2)
    g[:n2d, 2] = 0.0
    n = _unit_rows(g)
    n[0] = (1.0, 0.0, 0.0)
    if n_normals > 1:
        n[1] = (np.sqrt(0.5), np.sqrt(0.5), 0.0)
    n = n.astype(np.float32)
    v = (np.arange(L, dtype=np.float64) / max(L - 1, 1)).astype(np.float32)
    V0 = np.tile(v, n_normals)
    nx, ny, nz = (np.repeat(n[:, i], L) for i in range(3))
    return V0, nx, ny, nz


def roundtrip_volumes(L: int):
    """The L volumes plic_roundtrip_error steps through (include/plic.h): fp32 l*h with
    h = fp32(1/(L-1)), the last one exactly 1 (the paper's "equally spaced, edge cases
    included")."""
    h = np.float32(1.0) / np.float32(L - 1)
    v = np.arange(L, dtype=np.float32) * h
    v[L - 1] = np.float32(1.0)
    return v.astype(np.float32)


def paper_normals(n_normals: int, seed: int, workers=None):
    """The normal set of the paper's GPU test at any size: normal 0 is
    (1,0,0), normal 1 is (1/sqrt2, 1/sqrt2, 0), normals 2 .. n_normals/8 - 1 are random 2D
    directions in the x-y plane, the rest random 3D directions (67108864 normals in the
    paper: 8388606 2D, 58720256 3D).  Chunked like random_sphere.  Returns nx, ny, nz."""
    n2d = max(n_normals // 8, 2)

    def fn(c):
        g = _rng(seed, _STREAM_PAPER_NORMALS, c).standard_normal((CHUNK, 3))
        idx = c * CHUNK + np.arange(CHUNK)
        g[idx < n2d, 2] = 0.0
        n = _unit_rows(g)
        if c == 0:
            n[0] = (1.0, 0.0, 0.0)
            n[1] = (np.sqrt(0.5), np.sqrt(0.5), 0.0)
        return np.zeros(CHUNK, dtype=np.float32), n.astype(np.float32)

    _, nx, ny, nz = _run_chunks(fn, 0, n_normals, workers)
    return nx, ny, nz


def sphere_lattice(L: int = 256, R: float = 60.0, centre=(128.3, 127.7, 128.1), sub: int = 8):
    """Config 5: fill levels of a sphere on an L^3 lattice.  Cell (i,j,k) spans
    [i,i+1)x[j,j+1)x[k,k+1) with its centre at (i+1/2, j+1/2, k+1/2) (the paper does
    not fix the convention; this one is stated in DESIGN.md).  phi = fraction of the
    sub^3 sample points (sub-cell centres) with |p - centre| <= R.  Interface cells are
    those with 0 < phi < 1; their normal is (cell centre - sphere centre)/|.|, i.e. it
    points out of the fluid.  Returns a dict of arrays over the interface cells:
    phi, nx, ny, nz (fp32), r (fp64 distance of the cell centre from the sphere
    centre), ijk (int32 [M,3])."""
    o = np.asarray(centre, dtype=np.float64)
    half_diag = 0.5 * np.sqrt(3.0)
    offs = (np.arange(sub, dtype=np.float64) + 0.5) / sub
    sx, sy, sz = np.meshgrid(offs, offs, offs, indexing="ij")
    s = np.stack([sx.ravel(), sy.ravel(), sz.ravel()], axis=1)          # [sub^3, 3]
    ax = np.arange(L, dtype=np.float64)
    out_phi, out_n, out_r, out_ijk = [], [], [], []
    for i in range(L):
        cy, cz = np.meshgrid(ax + 0.5, ax + 0.5, indexing="ij")
        cx = np.full_like(cy, i + 0.5)
        r = np.sqrt((cx - o[0]) ** 2 + (cy - o[1]) ** 2 + (cz - o[2]) ** 2)
        shell = np.abs(r - R) <= half_diag + 1e-9
        if not shell.any():
            continue
        jj, kk = np.nonzero(shell)
        corner = np.stack([np.full(jj.shape, float(i)), jj.astype(np.float64),
                           kk.astype(np.float64)], axis=1)              # [m, 3]
        p = corner[:, None, :] + s[None, :, :] - o[None, None, :]       # [m, sub^3, 3]
        inside = np.einsum("msk,msk->ms", p, p) <= R * R
        phi = inside.mean(axis=1)
        itf = (phi > 0.0) & (phi < 1.0)
        if not itf.any():
            continue
        c = corner[itf] + 0.5 - o[None, :]
        rr = np.sqrt(np.einsum("ij,ij->i", c, c))
        out_phi.append(phi[itf])
        out_n.append(c / rr[:, None])
        out_r.append(rr)
        out_ijk.append(np.stack([np.full(itf.sum(), i), jj[itf], kk[itf]], axis=1))
    phi = np.concatenate(out_phi).astype(np.float32)
    n = np.concatenate(out_n).astype(np.float32)
    return {"phi": phi, "nx": n[:, 0].copy(), "ny": n[:, 1].copy(), "nz": n[:, 2].copy(),
            "r": np.concatenate(out_r), "ijk": np.concatenate(out_ijk).astype(np.int32),
            "R": float(R), "centre": tuple(float(x) for x in o)}


def sphere_fill_lattice(L: int = 256, R: float = 60.0, centre=(128.3, 127.7, 128.1), sub: int = 8):
    """Config 5 as a full lattice for plic_curvature: phi[z, y, x] (fp32, L^3), 1 inside the sphere,
    0 outside, and on the interface the sampled fraction of sphere_lattice() (same convention)."""
    cells = sphere_lattice(L, R, centre, sub)
    o = np.asarray(centre, dtype=np.float64)
    ax = np.arange(L, dtype=np.float64) + 0.5
    r2 = ((ax - o[2]) ** 2)[:, None, None] + ((ax - o[1]) ** 2)[None, :, None] + ((ax - o[0]) ** 2)[None, None, :]
    phi = (r2 < R * R).astype(np.float32)
    ijk = cells["ijk"]
    phi[ijk[:, 2], ijk[:, 1], ijk[:, 0]] = cells["phi"]
    return phi


def shard_range(N: int, rank: int, world: int, align: int = 32):
    """Contiguous [lo, hi) of N cells owned by `rank` of `world` ranks; interior
    boundaries are multiples of `align` cells so every shard keeps the 128-byte
    alignment of the parent arrays.  The union over ranks is exactly [0, N)."""
    if world <= 0 or not (0 <= rank < world):
        raise ValueError("bad rank/world")
    blocks = (N + align - 1) // align
    base, rem = divmod(blocks, world)
    lo_b = rank * base + min(rank, rem)
    hi_b = lo_b + base + (1 if rank < rem else 0)
    return min(lo_b * align, N), min(hi_b * align, N)
