"""CPU pins of the case-stratified workload generator (oracle/stratified.c, BASELINE.json configs[2]).

It is an input generator, not oracle arithmetic, but bench.py --gpus N hands each rank its own
`start`, and the parity tests label cells by its case output, so: the case mix is 20 % each, a cell
depends on (seed, index) only -- not on the chunk it is generated in, the thread count or the
layout -- and the label is the intersection case of eq. (11) that the oracle's own
classifier gives for the plane the oracle recovers from the returned (V0, n)."""
import numpy as np

import oracle
from oracle import stratified as st

N = 20000


def test_case_mix_is_one_fifth_each_and_inputs_are_in_domain():
    V0, nx, ny, nz, kase = st.stratified(N)
    assert all(a.dtype == np.float32 and a.shape == (N,) for a in (V0, nx, ny, nz)) and kase.dtype == np.int8
    assert np.array_equal(kase, (np.arange(N) % 5 + 1).astype(np.int8))       # cell i targets case i mod 5 + 1
    counts = np.bincount(kase, minlength=6)[1:]
    assert counts.tolist() == [N // 5] * 5
    assert np.all((V0 >= 0) & (V0 <= 1))
    norm = np.sqrt(nx.astype(np.float64) ** 2 + ny.astype(np.float64) ** 2 + nz.astype(np.float64) ** 2)
    assert np.all(np.abs(norm - 1) < 2e-7)
    # both halves of the cube and all eight octants of the normal occur in every case
    for k in range(1, 6):
        m = kase == k
        assert (V0[m] < 0.5).any() and (V0[m] > 0.5).any()
        assert len({(a > 0, b > 0, c > 0) for a, b, c in zip(nx[m][:400], ny[m][:400], nz[m][:400])}) == 8


def test_a_cell_depends_on_seed_and_index_only():
    whole = st.stratified(N, threads=1)
    for threads in (2, 5):
        again = st.stratified(N, threads=threads)
        assert all(np.array_equal(a, b) for a, b in zip(whole, again))
    # a shard generated with its own start (what a rank of bench.py --gpus N does), odd offset and length
    lo, hi = 6007, 13331
    part = st.stratified(hi - lo, start=lo, threads=3)
    assert all(np.array_equal(a[lo:hi], b) for a, b in zip(whole, part))
    # another seed is another stream
    other = st.stratified(N, seed=st.SEED + 1)
    assert not np.array_equal(whole[0], other[0]) and np.array_equal(whole[4], other[4])


def test_contiguous_layout_is_a_permutation_of_the_same_cells():
    a = st.stratified(N)
    for start in (0, 3):                                          # the gather honours the offset's residue
        a = st.stratified(N, start=start)
        c = st.stratified(N, start=start, contiguous=True)
        assert np.array_equal(c[4], np.repeat(np.arange(1, 6), N // 5).astype(np.int8))
        key = lambda t: np.lexsort((t[3], t[2], t[1], t[0], t[4]))
        ia, ic = key(a), key(c)
        assert all(np.array_equal(x[ia], y[ic]) for x, y in zip(a, c))


def test_labels_are_the_oracles_case_of_the_recovered_plane():
    V0, nx, ny, nz, kase = st.stratified(N)
    d0 = oracle.solve(V0, nx, ny, nz)
    # V0 is the fp32 rounding of the oracle's forward map at the drawn plane, so the recovered plane
    # reproduces it to fp32 rounding ...
    assert np.max(np.abs(oracle.volume(d0, nx, ny, nz) - V0.astype(np.float64))) < 1e-10
    # ... and lies in the labelled case, except where that rounding of V0 moved a plane drawn within
    # ~1e-7 of a case boundary across it
    got = oracle.case(d0, nx, ny, nz)
    differ = got != kase
    assert differ.mean() < 1e-3
    assert np.all(np.abs(got[differ].astype(int) - kase[differ].astype(int)) <= 2)
