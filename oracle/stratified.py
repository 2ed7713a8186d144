"""Case-stratified workload (BASELINE.json configs[2]) -- TEST / BENCH INFRASTRUCTURE.

Needs the oracle's case classifier and forward map (the config says "V0 computed by the oracle's
forward map"), so it is part of ``oracle/`` and not of ``gen/`` (which holds none of the method's
arithmetic).  The arithmetic and the counter-based random numbers are in ``oracle/stratified.c``;
this module only marshals.  Used by ``tests/`` (parity per case) and by ``bench.py``'s
``divergence`` leg (input generation only, outside every timed region).

Cell i targets intersection case (i mod 5) + 1; ``contiguous=True`` returns the same cells
gathered into five case-contiguous blocks (every warp then holds one case), the default
interleaving puts all five cases into every warp.
"""
from __future__ import annotations

import ctypes

import numpy as np

from . import _load

SEED = 2                  # BASELINE.json configs[2]


def stratified(N: int, seed: int = SEED, contiguous: bool = False, start: int = 0, threads: int = 0):
    """fp32 (V0, nx, ny, nz) and the int8 case label of the cells [start, start+N)."""
    lib = _load()
    fp = ctypes.POINTER(ctypes.c_float)
    fn = lib.oracle_stratified_cells
    fn.argtypes = [ctypes.c_uint64, ctypes.c_int64, ctypes.c_int64, fp, fp, fp, fp,
                   ctypes.POINTER(ctypes.c_int8), ctypes.c_int]
    fn.restype = ctypes.c_int64
    V0, nx, ny, nz = (np.empty(N, dtype=np.float32) for _ in range(4))
    kase = np.empty(N, dtype=np.int8)
    worst = fn(seed, start, N, *[a.ctypes.data_as(fp) for a in (V0, nx, ny, nz)],
               kase.ctypes.data_as(ctypes.POINTER(ctypes.c_int8)), threads)
    if worst < 0:
        raise RuntimeError("stratified generator: a cell found no draw of its case")
    if contiguous:
        # cell i has case (i mod 5) + 1: gather the five residue classes (a stable sort by case)
        order = np.concatenate([np.arange((k - start) % 5, N, 5) for k in range(5)])
        V0, nx, ny, nz, kase = V0[order], nx[order], ny[order], nz[order], kase[order]
    return V0, nx, ny, nz, kase
