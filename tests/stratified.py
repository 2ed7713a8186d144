"""Case-stratified workload (BASELINE.json configs[2]) -- test/bench infrastructure.

Needs the oracle's forward map and case classifier, so it lives with the tests and not in
gen/ (which holds none of the method's arithmetic).  Cell i targets intersection case
k = (i mod 5) + 1: draws (normal uniform on the sphere, d0 uniform on [-S/2, S/2]) are
repeated until the oracle classifies the plane as case k; V0 = fp32(oracle.volume(d0, n)).
Per-cell acceptance differs by case (about 26 / 33 / 18 / 4 / 18 %), so candidates are drawn
in bulk per Philox chunk and the first accepted candidate of each case is consumed in order.
`contiguous=True` returns the same cells sorted into five case-contiguous blocks (zero warp
divergence); the default interleaving puts all five cases into every warp.
"""
from __future__ import annotations

import numpy as np

import oracle

_STREAM_STRAT = 5
_CHUNK = 1 << 18          # cells per chunk (part of the recipe)
_OVERSAMPLE = 40          # candidates per cell of the rarest case (acceptance ~4 %)


def _chunk(seed: int, c: int):
    key = np.array([seed, _STREAM_STRAT], dtype=np.uint64)
    counter = np.array([0, 0, 0, c], dtype=np.uint64)
    rng = np.random.Generator(np.random.Philox(key=key, counter=counter))
    per_case = _CHUNK // 5 + 1
    m = per_case * _OVERSAMPLE
    g = rng.standard_normal((m, 3))
    n = (g / np.sqrt((g * g).sum(1))[:, None]).astype(np.float32)
    S = np.abs(n.astype(np.float64)).sum(1)
    d0 = ((rng.random(m) - 0.5) * S).astype(np.float32)
    kase = oracle.case(d0, n[:, 0], n[:, 1], n[:, 2])
    picks = []
    for k in range(1, 6):
        idx = np.nonzero(kase == k)[0]
        if idx.shape[0] < per_case:
            raise RuntimeError("stratified generator: not enough case-%d candidates" % k)
        picks.append(idx[:per_case])
    order = np.stack(picks, 1).ravel()[:_CHUNK]       # interleave: cell i -> case (i mod 5)+1
    n, d0 = n[order], d0[order]
    V0 = oracle.volume(d0, n[:, 0], n[:, 1], n[:, 2]).astype(np.float32)
    return V0, n, (np.arange(_CHUNK) % 5 + 1).astype(np.int8)


def stratified(N: int, seed: int = 2, contiguous: bool = False):
    """fp32 (V0, nx, ny, nz) and the int8 target case of each cell."""
    V0 = np.empty(N, np.float32)
    n = np.empty((N, 3), np.float32)
    kase = np.empty(N, np.int8)
    for c, lo in enumerate(range(0, N, _CHUNK)):
        hi = min(N, lo + _CHUNK)
        v, nn, kk = _chunk(seed, c)
        # keep the 5-periodic pattern across chunk boundaries: _CHUNK % 5 != 0
        shift = lo % 5
        if shift:
            v, nn, kk = np.roll(v, -shift), np.roll(nn, -shift, axis=0), np.roll(kk, -shift)
        V0[lo:hi], n[lo:hi], kase[lo:hi] = v[:hi - lo], nn[:hi - lo], kk[:hi - lo]
    if contiguous:
        order = np.argsort(kase, kind="stable")
        V0, n, kase = V0[order], n[order], kase[order]
    return V0, n[:, 0].copy(), n[:, 1].copy(), n[:, 2].copy(), kase
