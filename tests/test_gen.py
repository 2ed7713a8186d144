"""Host-side checks of the seeded workload generators (gen/): determinism, per-index
independence of N / offset / worker count, and the composition each config promises."""
import numpy as np

import gen


def test_random_sphere_deterministic_and_offset_independent():
    a = gen.random_sphere(3000, seed=7)
    b = gen.random_sphere(3000, seed=7, workers=1)
    for x, y in zip(a, b):
        assert x.dtype == np.float32 and np.array_equal(x, y)
    # a window straddling a chunk boundary equals the same cells of a longer run
    start = gen.CHUNK - 1000
    w = gen.random_sphere(2500, seed=7, start=start)
    full = gen.random_sphere(gen.CHUNK + 1500, seed=7, workers=2)
    for x, y in zip(w, full):
        assert np.array_equal(x, y[start:start + 2500])
    c = gen.random_sphere(3000, seed=8)
    assert not np.array_equal(a[0], c[0])


def test_random_sphere_distribution():
    V0, nx, ny, nz = gen.random_sphere(200000, seed=1)
    r = np.sqrt(nx.astype(np.float64) ** 2 + ny.astype(np.float64) ** 2 + nz.astype(np.float64) ** 2)
    assert np.max(np.abs(r - 1.0)) < 2e-7
    assert V0.min() >= 0.0 and V0.max() <= 1.0
    assert abs(V0.mean() - 0.5) < 5e-3
    for c in (nx, ny, nz):                       # uniform on the sphere: each component ~ U[-1,1]
        assert abs(c.mean()) < 5e-3 and abs(c.var() - 1.0 / 3.0) < 5e-3


def test_edge_cells_composition():
    V0, nx, ny, nz = gen.edge_cells(4096, seed=0)
    n = np.stack([nx, ny, nz], 1)
    zeros = (n == 0.0).sum(1)
    j = np.arange(4096)
    assert np.array_equal(zeros, np.where((j // 5) % 2 == 1, 2, 1))
    ones = np.abs(n[zeros == 2]).max(1)
    assert np.all(ones == 1.0)                   # single survivor is exactly +-1
    assert (n < 0).any() and (n > 0).any()
    assert np.array_equal(V0, gen.workloads.EDGE_V0[j % 5])
    assert set(np.unique(V0).tolist()) == {0.0, 0.5, 1.0, float(np.float32(1e-7)),
                                           float(np.float32(1.0 - 1e-7))}
    r = np.sqrt((n.astype(np.float64) ** 2).sum(1))
    assert np.max(np.abs(r - 1.0)) < 2e-7


def test_config1_layout():
    V0, nx, ny, nz = gen.config1(seed=0, n_random=5000, n_edge=100)
    assert V0.shape == (5100,)
    a = gen.random_sphere(5000, 0)
    assert np.array_equal(nx[:5000], a[1])
    assert np.array_equal(nz[5000:], gen.edge_cells(100, 0)[3])


def test_snapped_beta_composition():
    V0, nx, ny, nz = gen.snapped_beta(200000, seed=3)
    n = np.stack([nx, ny, nz], 1)
    zeros = (n == 0.0).sum(1)
    axis = zeros == 2
    diag = zeros == 1
    assert abs(axis.mean() - 0.25) < 5e-3 and abs(diag.mean() - 0.25) < 5e-3
    assert np.all(np.abs(n[axis]).max(1) == 1.0)
    d = np.abs(n[diag])
    assert np.all((d == 0.0) | (d == np.float32(0.70710677)))
    # Beta(1/2,1/2): mean 1/2, variance 1/8, mass near the ends
    assert abs(V0.mean() - 0.5) < 5e-3 and abs(V0.var() - 0.125) < 3e-3
    assert (V0 < 0.01).mean() > 0.05 and (V0 > 0.99).mean() > 0.05
    w = gen.snapped_beta(1000, seed=3, start=777)
    assert np.array_equal(w[2], ny[777:1777])


def test_paper_benchmark_set_shape():
    V0, nx, ny, nz = gen.paper_benchmark_set(64, 17, seed=5)
    assert V0.shape == (64 * 17,)
    assert V0[0] == 0.0 and V0[16] == 1.0
    assert (nx[0], ny[0], nz[0]) == (1.0, 0.0, 0.0)
    assert nz[17] == 0.0 and nx[17] == ny[17] == np.float32(np.sqrt(0.5))
    n2d = (nz.reshape(64, 17)[:, 0] == 0.0).sum()
    assert n2d == 8                               # 12.5 % 2-D normals incl. the two fixed ones


def test_sphere_lattice_small():
    s = gen.sphere_lattice(L=32, R=10.0, centre=(16.3, 15.7, 16.1), sub=4)
    assert s["phi"].min() > 0.0 and s["phi"].max() < 1.0
    m = s["phi"].shape[0]
    assert 1000 < m < 3000                        # ~ 4 pi R^2 * O(1) interface cells
    # interface cells hug the sphere; normals point away from the centre
    assert np.max(np.abs(s["r"] - 10.0)) <= 0.5 * np.sqrt(3) + 1e-9
    c = s["ijk"] + 0.5 - np.asarray(s["centre"])
    dots = (c * np.stack([s["nx"], s["ny"], s["nz"]], 1)).sum(1)
    assert np.allclose(dots, s["r"], rtol=1e-6)
    # total fluid volume of interface cells + full cells ~ sphere volume (coarse check)
    assert 0.2 < s["phi"].mean() < 0.8


def test_shard_range_partitions_exactly():
    for N in (0, 1, 31, 32, 33, 1000, (1 << 20) + 4096):
        for world in (1, 2, 3, 8):
            spans = [gen.shard_range(N, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == N
            for (a, b), (c, d) in zip(spans, spans[1:]):
                assert b == c and a <= b
            for lo, hi in spans[:-1]:
                assert hi % 32 == 0 or hi == N


def test_paper_normals_and_roundtrip_volumes():
    import gen
    nx, ny, nz = gen.paper_normals(4096, seed=9)
    assert nx.dtype == np.float32 and nx.shape == (4096,)
    assert (nx[0], ny[0], nz[0]) == (1.0, 0.0, 0.0)
    assert abs(nx[1] - np.sqrt(0.5)) < 1e-7 and abs(ny[1] - np.sqrt(0.5)) < 1e-7 and nz[1] == 0.0
    assert np.all(nz[:512] == 0.0) and np.count_nonzero(nz[512:] == 0.0) == 0    # 12.5 % 2-D normals
    assert np.max(np.abs(nx.astype(np.float64) ** 2 + ny.astype(np.float64) ** 2 + nz.astype(np.float64) ** 2 - 1)) < 3e-7
    again = gen.paper_normals(4096, seed=9)
    assert all(np.array_equal(a, b) for a, b in zip((nx, ny, nz), again))
    v = gen.roundtrip_volumes(256)
    assert v.dtype == np.float32 and v[0] == 0.0 and v[-1] == 1.0 and np.all(np.diff(v) > 0)
    assert np.max(np.abs(v - np.arange(256) / 255.0)) < 1e-7
    assert gen.roundtrip_volumes(2).tolist() == [0.0, 1.0]


def test_sphere_fill_lattice():
    import gen
    phi = gen.sphere_fill_lattice(32, 10.0, (16.3, 15.7, 16.1), 8)
    assert phi.shape == (32, 32, 32) and phi.dtype == np.float32
    assert phi.min() == 0.0 and phi.max() == 1.0
    assert abs(phi.sum() - 4.0 / 3.0 * np.pi * 1000.0) < 5.0              # the drop's volume
    itf = (phi > 0) & (phi < 1)
    z, y, x = np.nonzero(itf)
    r = np.sqrt((x + 0.5 - 16.3) ** 2 + (y + 0.5 - 15.7) ** 2 + (z + 0.5 - 16.1) ** 2)
    assert np.all(np.abs(r - 10.0) <= 0.5 * np.sqrt(3.0) + 1e-9)         # interface cells straddle the sphere
    assert np.all(np.round(phi[itf] * 512) == phi[itf] * 512)            # fractions of 8^3 points
