"""GPU parity: the CUDA path (through the C ABI of libplic) against the fp64 CPU oracle,
element by element on the same seeded inputs.

Bars (BASELINE.json north_star): |d0 - d0_ref| <= 2e-5 absolute; forward-volume residual
|V0_oracle(d0_gpu, n) - V0| <= 2e-5; finite everywhere, including n1 = 0, n1 = n2 = 0 and
V0 in {0, 1/2, 1}.  plic_volume: |V0 - V0_ref| <= 1e-6 (DESIGN.md derives it from fp32
rounding of the stable forms).  All eight plic_solve variants (4 methods x precise/fast).
"""
import os
import sys

import numpy as np
import pytest
import torch

import gen
import oracle

from oracle.stratified import stratified

pytestmark = pytest.mark.gpu

TOL_D0 = 2e-5        # north_star
TOL_RES = 2e-5       # north_star
TOL_VOL = 1e-6

VARIANTS = [(m, f) for m in ("analytic", "sz", "newton", "nested") for f in (False, True)]
IDS = ["%s%s" % (m, "-fast" if f else "") for m, f in VARIANTS]


@pytest.fixture(scope="module")
def plic():
    import paper_2006_12838_b200 as p
    assert os.path.exists(p.LIB_PATH)
    return p


def dev(*arrays):
    return [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrays]


def check_solve(plic, V0, nx, ny, nz, method, fast, ref=None, what=""):
    tV, tx, ty, tz = dev(V0, nx, ny, nz)
    before = plic.plic_launch_count()
    d0 = plic.plic_solve(tV, tx, ty, tz, method=method, fast=fast)
    torch.cuda.synchronize()
    assert plic.plic_launch_count() > before or len(V0) == 0     # the CUDA path ran
    got = d0.cpu().numpy()
    assert got.dtype == np.float32 and got.shape == V0.shape
    assert np.all(np.isfinite(got)), "%s: non-finite d0" % what
    if ref is None:
        ref = oracle.solve(V0, nx, ny, nz)
    err = np.abs(got.astype(np.float64) - ref)
    i = int(np.argmax(err)) if len(err) else 0
    assert err.max(initial=0.0) <= TOL_D0, "%s: |d0-ref| max %.3e at cell %d (V0=%r n=%r got=%r ref=%r)" % (
        what, err.max(), i, V0[i], (nx[i], ny[i], nz[i]), got[i], ref[i])
    res = np.abs(oracle.volume(got, nx, ny, nz) - np.clip(V0.astype(np.float64), 0.0, 1.0))
    assert res.max(initial=0.0) <= TOL_RES, "%s: residual max %.3e" % (what, res.max())
    S2 = 0.5 * (np.abs(nx.astype(np.float64)) + np.abs(ny) + np.abs(nz))
    assert np.all(np.abs(got) <= S2 * (1 + 1e-6) + 1e-7)           # eq. (1): d0 in [-S/2, S/2]
    return got, err


# ------------------------------------------------------------------------------------------
# config 1: 2^20 random + 4096 edge cells, seed 0, all variants
# ------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def config1():
    V0, nx, ny, nz = gen.config1(seed=0)
    return V0, nx, ny, nz, oracle.solve(V0, nx, ny, nz)


@pytest.mark.parametrize("method,fast", VARIANTS, ids=IDS)
def test_config1_all_cells(plic, config1, method, fast):
    V0, nx, ny, nz, ref = config1
    assert V0.shape[0] == (1 << 20) + 4096
    got, err = check_solve(plic, V0, nx, ny, nz, method, fast, ref, "config1")
    edge = slice(1 << 20, None)
    assert err[edge].max() <= TOL_D0
    # exact volumes on the edge cells: V0 = 0 / 1 are the ends of the interval, 1/2 its centre
    S2 = 0.5 * (np.abs(nx[edge]) + np.abs(ny[edge]) + np.abs(nz[edge])).astype(np.float64)
    v = V0[edge]
    assert np.max(np.abs(got[edge][v == 0.0] + S2[v == 0.0])) <= 2e-7
    assert np.max(np.abs(got[edge][v == 1.0] - S2[v == 1.0])) <= 2e-7
    assert np.max(np.abs(got[edge][v == 0.5])) <= 2e-7


@pytest.mark.parametrize("method,fast", VARIANTS, ids=IDS)
def test_config1_observed_error_regression(plic, config1, method, fast):
    """Not the parity bar (that is TOL_D0 = 2e-5, above) but a regression guard on what DESIGN.md
    reports as observed: on configs[0] the precise kernels stay within 3.2e-7 of the oracle and the fast
    ones within 8.2e-7 (round-2 measurement: analytic 1.8e-7 / 3.8e-7, SZ 3.2e-7 / 8.2e-7, Newton
    1.5e-7 / 1.7e-7, nested 1.6e-7 / 2.9e-7; a few fp32 ulp of an offset <= 0.87).  A change that
    costs accuracy (an iteration dropped, a coarser polynomial) trips this long before 2e-5."""
    V0, nx, ny, nz, ref = config1
    got = plic.plic_solve(*dev(V0, nx, ny, nz), method=method, fast=fast).cpu().numpy()
    err = np.abs(got.astype(np.float64) - ref)
    if method == "nested" and fast:
        # round 3: 16 fixed halvings instead of 20 (14 halvings give
        # 1.2e-5, 20 give 2.9e-7).  The centre after 16 halvings is within w 2^-17 <= 0.577 * 2^-17 =
        # 4.4e-6 of the root (w = bracket width <= n1), plus fp32 rounding; the parity bar stays 2e-5.
        assert err.max() <= 4.8e-6, err.max()
        assert err.mean() <= 1.0e-6, err.mean()
        return
    assert err.max() <= (1.5e-6 if fast else 6e-7), err.max()
    assert err.mean() <= (1.5e-7 if fast else 6e-8), err.mean()


# ------------------------------------------------------------------------------------------
# ragged sizes, misaligned pointers, aliasing, empty input
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("method,fast", VARIANTS, ids=IDS)
def test_ragged_and_misaligned(plic, method, fast):
    V0, nx, ny, nz = gen.random_sphere(70001, seed=11)
    ref = oracle.solve(V0, nx, ny, nz)
    tV, tx, ty, tz = dev(V0, nx, ny, nz)
    for N in (0, 1, 2, 3, 4, 5, 7, 255, 256, 1023, 1027, 65537, 70001):
        out = plic.plic_solve(tV[:N], tx[:N], ty[:N], tz[:N], method=method, fast=fast)
        assert out.shape == (N,)
        if N:
            assert np.max(np.abs(out.cpu().numpy().astype(np.float64) - ref[:N])) <= TOL_D0
    # common misalignment (head cells), offsets 1..3 floats
    for off in (1, 2, 3):
        N = 4099
        out = torch.full((off + N + 5,), 7.0, device="cuda")
        plic.plic_solve(tV[off:off + N], tx[off:off + N], ty[off:off + N], tz[off:off + N],
                        out=out[off:off + N], method=method, fast=fast)
        got = out.cpu().numpy()
        assert np.all(got[:off] == 7.0) and np.all(got[off + N:] == 7.0)      # no overrun
        assert np.max(np.abs(got[off:off + N].astype(np.float64) - ref[off:off + N])) <= TOL_D0
    # mixed misalignment: scalar path for the whole range
    N = 5001
    out = plic.plic_solve(tV[1:1 + N], tx[2:2 + N].clone()[0:N], ty[3:3 + N], tz[0:N],
                          method=method, fast=fast)
    ref_mixed = oracle.solve(V0[1:1 + N], nx[2:2 + N], ny[3:3 + N], nz[0:N])
    assert np.max(np.abs(out.cpu().numpy().astype(np.float64) - ref_mixed)) <= TOL_D0
    # d0 may alias V0
    a = tV.clone()
    plic.plic_solve(a, tx, ty, tz, out=a, method=method, fast=fast)
    assert np.max(np.abs(a.cpu().numpy().astype(np.float64) - ref)) <= TOL_D0


def test_vector_and_scalar_paths_agree_bitwise(plic):
    V0, nx, ny, nz = gen.random_sphere(50000, seed=12)
    tV, tx, ty, tz = dev(V0, nx, ny, nz)
    for method, fast in VARIANTS:
        a = plic.plic_solve(tV, tx, ty, tz, method=method, fast=fast)
        # force the scalar kernel: give one input a different alignment
        sx = torch.empty(50001, device="cuda")[1:]
        sx.copy_(tx)
        b = plic.plic_solve(tV, sx, ty, tz, method=method, fast=fast)
        assert torch.equal(a, b), (method, fast)


# ------------------------------------------------------------------------------------------
# the paper's own benchmark shape: axis normal, face diagonal, 12.5 % 2-D normals,
# V0 equally spaced including 0 and 1; round-trip error of eq. (31)-(32)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("method,fast", VARIANTS, ids=IDS)
def test_paper_benchmark_set_and_round_trip(plic, method, fast):
    V0, nx, ny, nz = gen.paper_benchmark_set(2048, 257, seed=5)
    got, _ = check_solve(plic, V0, nx, ny, nz, method, fast, None, "paper set")
    # the Kawano NaN cells: n = (1,0,0), V0 in {0,1}
    assert got[0] == -0.5 and got[256] == 0.5
    tV, tx, ty, tz = dev(V0, nx, ny, nz)
    back = plic.plic_volume(plic.plic_solve(tV, tx, ty, tz, method=method, fast=fast), tx, ty, tz)
    E = (back - tV).abs()
    # eq. (32): fp32 solvers reach E_avg of 2e-8 .. 7e-8 (Tables 1, 3); fast variants a bit above
    assert float(E.mean()) < (3e-7 if fast else 1e-7), float(E.mean())
    assert float(E.max()) < 2e-5


# ------------------------------------------------------------------------------------------
# config 3 shape: case-stratified, interleaved and case-contiguous
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("contiguous", [False, True], ids=["interleaved", "contiguous"])
def test_case_stratified(plic, contiguous):
    V0, nx, ny, nz, kase = stratified(1 << 19, seed=2, contiguous=contiguous)
    ref = oracle.solve(V0, nx, ny, nz)
    for method, fast in VARIANTS:
        _, err = check_solve(plic, V0, nx, ny, nz, method, fast, ref, "stratified")
        for k in range(1, 6):
            assert (kase == k).sum() > 100000 and err[kase == k].max() <= TOL_D0


# ------------------------------------------------------------------------------------------
# config 4 shape: snapped normals (exact zeros, equal components), V0 ~ Beta(1/2,1/2)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("method,fast", VARIANTS, ids=IDS)
def test_snapped_beta(plic, method, fast):
    V0, nx, ny, nz = gen.snapped_beta(1 << 20, seed=3)
    check_solve(plic, V0, nx, ny, nz, method, fast, None, "snapped")


# ------------------------------------------------------------------------------------------
# tiny smallest components: the regime where naive cubic arithmetic loses all digits
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("method,fast", VARIANTS, ids=IDS)
def test_small_n1_sweep(plic, method, fast):
    rng = np.random.default_rng(99)
    m = 1 << 17
    n1 = 10.0 ** rng.uniform(-12, -0.5, m)
    ang = rng.uniform(0, 2 * np.pi, m)
    g = np.stack([n1, np.cos(ang), np.sin(ang)], 1)
    g /= np.linalg.norm(g, axis=1, keepdims=True)
    perm = rng.permuted(np.tile(np.arange(3), (m, 1)), axis=1)
    g = np.take_along_axis(g, perm, 1).astype(np.float32)
    V0 = rng.random(m).astype(np.float32)
    check_solve(plic, V0, g[:, 0].copy(), g[:, 1].copy(), g[:, 2].copy(), method, fast, None, "small n1")


@pytest.mark.parametrize("method,fast", VARIANTS, ids=IDS)
def test_degenerate_inputs(plic, method, fast):
    s = np.float32(np.sqrt(0.5))
    t = np.float32(1.0 / np.sqrt(3.0))
    normals = [(1, 0, 0), (0, -1, 0), (0, 0, 1), (s, s, 0), (0, -s, s), (s, 0, -s), (t, t, t),
               (-t, t, -t), (0.6, 0.8, 0), (0, 0, 0), (1e-30, 0.6, 0.8), (1e-20, 1e-20, 1),
               (1e-38, 1e-38, 1), (3e-39, 0.6, 0.8), (2.0, 0.0, 0.0), (0.3, 0.4, 1.2)]
    vols = [0.0, 0.5, 1.0, 1e-7, 1 - 1e-7, 1e-30, 0.25, 0.75, 1.0 / 6.0, -0.5, 1.5]
    n = np.array([nn for nn in normals for _ in vols], dtype=np.float32)
    V0 = np.array([v for _ in normals for v in vols], dtype=np.float32)
    nx, ny, nz = n[:, 0].copy(), n[:, 1].copy(), n[:, 2].copy()
    ref = oracle.solve(V0, nx, ny, nz)              # oracle: V0<0 -> -S/2, V0>1 -> +S/2, n=0 -> 0
    tV, tx, ty, tz = dev(V0, nx, ny, nz)
    got = plic.plic_solve(tV, tx, ty, tz, method=method, fast=fast).cpu().numpy()
    assert np.all(np.isfinite(got))
    assert np.max(np.abs(got.astype(np.float64) - ref)) <= TOL_D0
    zero = (n == 0).all(1)
    assert np.all(got[zero] == 0.0)


def test_homogeneity_and_method_agreement(plic):
    V0, nx, ny, nz = gen.random_sphere(1 << 18, seed=21)
    tV, tx, ty, tz = dev(V0, nx, ny, nz)
    base = {}
    for method, fast in VARIANTS:
        d = plic.plic_solve(tV, tx, ty, tz, method=method, fast=fast)
        base[(method, fast)] = d
        for lam in (0.5, 4.0):                      # exact powers of two: d0(V0, c n) = c d0(V0, n)
            dl = plic.plic_solve(tV, tx * lam, ty * lam, tz * lam, method=method, fast=fast)
            assert float((dl - lam * d).abs().max()) <= 2e-5 * lam, (method, fast, lam)
    # "apart from floating-point errors, the SZ solution and our own produce identical
    # results"
    assert float((base[("analytic", False)] - base[("sz", False)]).abs().max()) <= 5e-6
    for key, d in base.items():
        assert float((d - base[("analytic", False)]).abs().max()) <= 2e-5, key


# ------------------------------------------------------------------------------------------
# forward map
# ------------------------------------------------------------------------------------------
def test_volume_parity(plic):
    V0, nx, ny, nz = gen.config1(seed=0)
    S = (np.abs(nx) + np.abs(ny) + np.abs(nz)).astype(np.float64)
    rng = np.random.default_rng(7)
    d0 = ((rng.random(V0.shape[0]) - 0.5) * S * 1.05).astype(np.float32)   # some planes miss the cube
    ref = oracle.volume(d0, nx, ny, nz)
    td, tx, ty, tz = dev(d0, nx, ny, nz)
    got = plic.plic_volume(td, tx, ty, tz).cpu().numpy()
    assert np.all(np.isfinite(got)) and got.min() >= 0.0 and got.max() <= 1.0
    assert np.max(np.abs(got.astype(np.float64) - ref)) <= TOL_VOL
    # ragged sizes and the zero normal
    for N in (1, 3, 5, 1027):
        g = plic.plic_volume(td[:N], tx[:N], ty[:N], tz[:N]).cpu().numpy()
        assert np.max(np.abs(g.astype(np.float64) - ref[:N])) <= TOL_VOL
    z = torch.zeros(3, device="cuda")
    g = plic.plic_volume(torch.tensor([-0.1, 0.0, 0.1], device="cuda"), z, z, z).cpu().numpy()
    assert g.tolist() == [0.0, 0.5, 1.0]


def test_volume_small_n1(plic):
    rng = np.random.default_rng(5)
    m = 1 << 17
    n1 = 10.0 ** rng.uniform(-12, -0.5, m)
    ang = rng.uniform(0, 2 * np.pi, m)
    g = np.stack([np.cos(ang), n1, np.sin(ang)], 1)
    g = (g / np.linalg.norm(g, axis=1, keepdims=True)).astype(np.float32)
    S = np.abs(g.astype(np.float64)).sum(1)
    d0 = ((rng.random(m) - 0.5) * S).astype(np.float32)
    ref = oracle.volume(d0, g[:, 0], g[:, 1], g[:, 2])
    td, tx, ty, tz = dev(d0, g[:, 0], g[:, 1], g[:, 2])
    got = plic.plic_volume(td, tx, ty, tz).cpu().numpy()
    assert np.max(np.abs(got.astype(np.float64) - ref)) <= TOL_VOL


# ------------------------------------------------------------------------------------------
# host-array API (the e2e path of bench.py)
# ------------------------------------------------------------------------------------------
def test_host_api_matches_device_api_bitwise(plic):
    N = (1 << 23) + 12345            # spans three pipeline chunks and a ragged tail
    V0, nx, ny, nz = gen.random_sphere(N, seed=31)
    tV, tx, ty, tz = dev(V0, nx, ny, nz)
    for method, fast in (("analytic", True), ("sz", False)):
        want = plic.plic_solve(tV, tx, ty, tz, method=method, fast=fast).cpu().numpy()
        got = plic.plic_solve_host(V0, nx, ny, nz, method=method, fast=fast)       # pageable numpy
        assert np.array_equal(got, want)
        pin = [torch.from_numpy(a).pin_memory() for a in (V0, nx, ny, nz)]
        out = torch.empty(N, dtype=torch.float32).pin_memory()
        plic.plic_solve_host(*pin, out=out, method=method, fast=fast)              # pinned torch
        assert np.array_equal(out.numpy(), want)
    d0 = plic.plic_solve(tV, tx, ty, tz).cpu().numpy()
    want = plic.plic_volume(*dev(d0, nx, ny, nz)).cpu().numpy()
    assert np.array_equal(plic.plic_volume_host(d0, nx, ny, nz), want)
    plic.plic_host_release()
    assert np.array_equal(plic.plic_volume_host(d0[:1000], nx[:1000], ny[:1000], nz[:1000]), want[:1000])


def test_non_default_stream(plic):
    V0, nx, ny, nz = gen.random_sphere(100000, seed=41)
    tV, tx, ty, tz = dev(V0, nx, ny, nz)
    want = plic.plic_solve(tV, tx, ty, tz, method="sz")
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        got = plic.plic_solve(tV, tx, ty, tz, method="sz")
    s.synchronize()
    assert torch.equal(got, want)


# ------------------------------------------------------------------------------------------
# full size, in the launch configuration bench.py times: 2^26 cells, seed 1; every 64th cell
# checked against the oracle, plus properties that hold at any size
# ------------------------------------------------------------------------------------------
def test_full_size_config2_sampled(plic):
    N = 1 << 26
    V0, nx, ny, nz = gen.random_sphere(N, seed=1)
    tV, tx, ty, tz = dev(V0, nx, ny, nz)
    sl = slice(5, None, 64)
    ref = oracle.solve(V0[sl], nx[sl], ny[sl], nz[sl])
    S2 = 0.5 * (tx.abs() + ty.abs() + tz.abs())
    out = torch.empty_like(tV)
    for method, fast in VARIANTS:
        grid, block, cpt = plic.plic_launch_config(method, N, fast)
        assert block == 256 and cpt == 4
        # one block per tile of 1024 cells (map_vec4) or per two tiles (map_tma)
        assert grid in (N // 1024, N // 2048)
        plic.plic_solve(tV, tx, ty, tz, out=out, method=method, fast=fast)
        assert bool(torch.isfinite(out).all())
        assert bool((out.abs() <= S2 * (1 + 1e-6)).all())
        assert bool((torch.sign(out) * torch.sign(tV - 0.5) >= 0).all())       # eq. (8)
        got = out[sl].cpu().numpy().astype(np.float64)
        assert np.max(np.abs(got - ref)) <= TOL_D0, (method, fast)
        back = plic.plic_volume(out, tx, ty, tz)
        assert float((back - tV).abs().max()) <= 2e-5                          # eq. (31)


def test_full_size_config3_sampled(plic):
    """configs[2] at its full size, in the layouts bench.py's `divergence` leg times: N = 2^26 cells
    labelled by the oracle, 20 % per intersection case, interleaved (every warp holds all five cases) and
    gathered into five case-contiguous blocks.  Properties on every cell, the oracle on every 64th cell
    with the error per case; both layouts hold the same cells, so their results agree bitwise after the
    gather."""
    N = 1 << 26
    V0, nx, ny, nz, kase = stratified(N, seed=2)
    assert np.all(np.abs(np.bincount(kase, minlength=6)[1:] - N / 5) <= 1)
    order = np.concatenate([np.arange(k, N, 5) for k in range(5)])
    sl = slice(3, None, 64)
    ref = oracle.solve(V0[sl], nx[sl], ny[sl], nz[sl])
    tV, tx, ty, tz = dev(V0, nx, ny, nz)
    torder = torch.from_numpy(order).cuda()
    cV, cx, cy, cz = [t[torder].contiguous() for t in (tV, tx, ty, tz)]
    S2 = 0.5 * (tx.abs() + ty.abs() + tz.abs())
    out, outc = torch.empty_like(tV), torch.empty_like(tV)
    for method, fast in VARIANTS:
        plic.plic_solve(tV, tx, ty, tz, out=out, method=method, fast=fast)
        plic.plic_solve(cV, cx, cy, cz, out=outc, method=method, fast=fast)
        assert bool(torch.isfinite(out).all()) and bool((out.abs() <= S2 * (1 + 1e-6)).all())
        assert bool(torch.equal(out[torder], outc)), (method, fast)              # layout independent
        err = np.abs(out[sl].cpu().numpy().astype(np.float64) - ref)
        for k in range(1, 6):
            assert err[kase[sl] == k].max() <= TOL_D0, (method, fast, k)
        back = plic.plic_volume(out, tx, ty, tz)
        assert float((back - tV).abs().max()) <= 2e-5                          # eq. (31)


def test_cuda_graph_capture_and_replay(plic):
    """The device-pointer calls only enqueue on the caller's stream (no synchronisation, no allocation), so a
    chain solve -> forward map -> solve can be captured into a CUDA graph and replayed on new data:
    the replay must equal the eager chain bitwise (programmatic dependent launches included)."""
    N = (1 << 20) + 77
    a = dev(*gen.random_sphere(N, seed=11))
    b = dev(*gen.random_sphere(N, seed=12))
    buf = [t.clone() for t in a]
    d0, V1, d1 = (torch.empty(N, dtype=torch.float32, device="cuda") for _ in range(3))

    def chain():
        plic.plic_solve(*buf, out=d0, method="analytic", fast=True)
        plic.plic_volume(d0, *buf[1:], out=V1)
        plic.plic_solve(V1, *buf[1:], out=d1, method="newton", fast=False)

    chain()
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        chain()
    for src in (b, a):
        for t, s_ in zip(buf, src):
            t.copy_(s_)
        g.replay()
        torch.cuda.synchronize()
        got = (d0.clone(), V1.clone(), d1.clone())
        chain()
        torch.cuda.synchronize()
        for x, y in zip(got, (d0, V1, d1)):
            assert bool(torch.equal(x, y))
    assert float((V1 - buf[0]).abs().max()) <= 2e-5


def test_more_than_2_31_cells(plic):
    """Maximum sizes: N = 2^31 + 2^20 + 5 cells (8.6 GB per array), beyond 32-bit element indices and with
    a ragged tail.  The input is a 2^22-cell block of configs[1] tiled on the device, so the expected
    output is the block's own result tiled: compared bitwise, chunk by chunk, for one kernel of each
    streaming body (map_tma, map_vec4, map_compact) and plic_volume.  Skipped when the device has less
    than 60 GB free."""
    free, _ = torch.cuda.mem_get_info()
    if free < 60 * (1 << 30):
        pytest.skip("needs 60 GB of free device memory")
    B = 1 << 22
    N = (1 << 31) + (1 << 20) + 5
    reps = (N + B - 1) // B
    base = dev(*gen.random_sphere(B, seed=1))
    big = [t.repeat(reps)[:N].contiguous() for t in base]
    out = torch.empty(N, dtype=torch.float32, device="cuda")
    for method, fast in (("analytic", True), ("nested", True), ("analytic", False)):
        want = plic.plic_solve(*base, method=method, fast=fast)
        out.fill_(float("nan"))
        plic.plic_solve(*big, out=out, method=method, fast=fast)
        full = (N // B) * B
        assert bool(torch.equal(out[:full].view(-1, B), want.expand(N // B, B))), (method, fast)
        assert bool(torch.equal(out[full:], want[:N - full])), (method, fast)
    want = plic.plic_volume(base[0], *base[1:])                  # any d0 in range will do: reuse V0 as d0
    plic.plic_volume(big[0], *big[1:], out=out)
    assert bool(torch.equal(out[:(N // B) * B].view(-1, B), want.expand(N // B, B)))
    assert bool(torch.equal(out[(N // B) * B:], want[:N - (N // B) * B]))
    del big, out
    torch.cuda.empty_cache()


def test_full_size_config4_sampled(plic):
    """configs[3]: N = 2^28 cells (4.3 GB in, 1.1 GB out), half the normals snapped to an axis or a
    face diagonal, V0 ~ Beta(1/2, 1/2): properties on every cell, the oracle on every 1024th."""
    N = 1 << 28
    V0, nx, ny, nz = gen.snapped_beta(N, seed=3)
    tV, tx, ty, tz = dev(V0, nx, ny, nz)
    sl = slice(7, None, 1024)
    ref = oracle.solve(V0[sl], nx[sl], ny[sl], nz[sl])
    S2 = 0.5 * (tx.abs() + ty.abs() + tz.abs())
    out = torch.empty_like(tV)
    for method, fast in (("analytic", True), ("sz", True), ("newton", True), ("nested", True), ("analytic", False)):
        plic.plic_solve(tV, tx, ty, tz, out=out, method=method, fast=fast)
        assert bool(torch.isfinite(out).all())
        assert bool((out.abs() <= S2 * (1 + 1e-6)).all())
        got = out[sl].cpu().numpy().astype(np.float64)
        assert np.max(np.abs(got - ref)) <= TOL_D0, (method, fast)
    back = plic.plic_volume(out, tx, ty, tz)
    assert float((back - tV).abs().max()) <= 2e-5                              # eq. (31)


# ------------------------------------------------------------------------------------------
# config 5: sphere of radius 60 on a 256^3 lattice
# ------------------------------------------------------------------------------------------
def test_sphere_lattice(plic):
    s = gen.sphere_lattice()
    phi, nx, ny, nz, r = s["phi"], s["nx"], s["ny"], s["nz"], s["r"]
    assert 55000 < phi.shape[0] < 65000
    ref = oracle.solve(phi, nx, ny, nz)
    dev_ref = np.abs(r + ref - 60.0)                # distance of the oracle's plane from the centre
    for method, fast in VARIANTS:
        got, _ = check_solve(plic, phi, nx, ny, nz, method, fast, ref, "sphere")
        dev_gpu = np.abs(r + got.astype(np.float64) - 60.0)
        # the reconstructed planes are as close to the sphere as the exact solver's: the
        # statistic is a property of the 8^3 fill-level sampler, not of the solver
        assert abs(dev_gpu.max() - dev_ref.max()) <= 4e-5
        assert abs(dev_gpu.mean() - dev_ref.mean()) <= 1e-5
        assert np.quantile(dev_gpu, 0.999) <= 0.05
        # BASELINE.json's literal "<= 0.05 cell" bound is exceeded by the exact fp64 solve on
        # a handful of nearly axis-aligned cells; the GPU must not add to them
        n_ref = int((dev_ref > 0.05).sum())
        assert n_ref <= 8
        assert (dev_gpu > 0.05 + 4e-5).sum() <= n_ref <= (dev_gpu > 0.05 - 4e-5).sum()


# ------------------------------------------------------------------------------------------
# plic_roundtrip_error: the paper's benchmark loop (sect. 2.6, eq. (31)-(33))
# ------------------------------------------------------------------------------------------
RT_VARIANTS = VARIANTS + [("blank", False)]
RT_IDS = IDS + ["blank"]


def _composed_roundtrip(plic, nx, ny, nz, L, method, fast):
    """eq. (31) assembled from the two parity-tested entry points, with the summation order
    include/plic.h states (fp32; even l and odd l separately, then added)."""
    n = len(nx)
    v = gen.roundtrip_volumes(L)
    V0 = np.tile(v, n)
    ax, ay, az = (np.repeat(a, L) for a in (nx, ny, nz))
    tV, tx, ty, tz = dev(V0, ax, ay, az)
    if method == "blank":
        d0 = tV - 0.5                                                   # eq. (33), exact in fp32
    else:
        d0 = plic.plic_solve(tV, tx, ty, tz, method=method, fast=fast)
    V = plic.plic_volume(d0, tx, ty, tz)
    err = (V - tV).abs().cpu().numpy().reshape(n, L)
    acc = np.zeros((n, 2), dtype=np.float32)
    for l in range(L):
        acc[:, l & 1] += err[:, l]
    return (acc[:, 0] + acc[:, 1]) / np.float32(L), d0.cpu().numpy().reshape(n, L)


@pytest.mark.parametrize("L", [256, 17, 2])
@pytest.mark.parametrize("method,fast", RT_VARIANTS, ids=RT_IDS)
def test_roundtrip_error_kernel(plic, method, fast, L):
    n = 3001
    nx, ny, nz = gen.paper_normals(n, seed=21)         # (1,0,0), face diagonal, 2-D, 3-D normals
    tx, ty, tz = dev(nx, ny, nz)
    before = plic.plic_launch_count()
    E = plic.plic_roundtrip_error(tx, ty, tz, L, method=method, fast=fast).cpu().numpy()
    assert plic.plic_launch_count() == before + 1
    assert E.shape == (n,) and np.all(np.isfinite(E))                   # no NaN at n = (1,0,0), V0 in {0,1}
    # (a) the fused loop equals the composition of plic_solve and plic_volume (both held to the
    #     oracle above); the few-ulp slack covers fused-multiply-add contraction differences
    E_comp, d0 = _composed_roundtrip(plic, nx, ny, nz, L, method, fast)
    assert np.max(np.abs(E - E_comp)) <= 2e-8, np.max(np.abs(E - E_comp))
    # (b) against the oracle: the fp64 round trip is exact (pinned to 1e-12), so E is the
    #     method's forward-volume residual, bounded as in north_star
    v = gen.roundtrip_volumes(L).astype(np.float64)
    if method == "blank":
        ax, ay, az = (np.repeat(a, L) for a in (nx, ny, nz))
        ref = np.abs(oracle.volume((np.tile(v, n) - 0.5).astype(np.float32), ax, ay, az) - np.tile(v, n))
        E_ref = ref.reshape(n, L).mean(axis=1)
        assert np.max(np.abs(E - E_ref)) <= TOL_VOL
    else:
        assert E.max() <= TOL_RES
        # fp32 error scale of Tables 1 and 3 (2e-8 .. 7e-8): same order here
        assert E.astype(np.float64).mean() <= 3e-7, E.mean()


def test_roundtrip_error_empty_and_validation(plic):
    tx = torch.zeros(0, device="cuda")
    assert plic.plic_roundtrip_error(tx, tx, tx, 8).shape == (0,)
    t = torch.ones(4, device="cuda")
    with pytest.raises(plic.PlicError):
        plic.plic_roundtrip_error(t, t, t, 1)


# ------------------------------------------------------------------------------------------
# PLIC_METHOD_KAWANO: Listing 3 as translated from Kawano's Fortran -- the paper's fifth variant
# ------------------------------------------------------------------------------------------
def test_kawano_reproduces_the_papers_nan_and_agrees_elsewhere(plic):
    # (a) the defect the paper reports: n = (1,0,0), V0 in {0, 1} -> NaN,
    #     which turns E_avg of the benchmark set into NaN (Tables 1-3: "-NaN")
    V0 = np.array([0.0, 1.0, 0.0, 1.0, 0.0, 1.0], dtype=np.float32)
    nx = np.array([1, 1, 0, 0, 0, 0], dtype=np.float32)
    ny = np.array([0, 0, -1, -1, 0, 0], dtype=np.float32)
    nz = np.array([0, 0, 0, 0, 1, 1], dtype=np.float32)
    got = plic.plic_solve(*dev(V0, nx, ny, nz), method="kawano").cpu().numpy()
    assert np.all(np.isnan(got))
    for m, f in VARIANTS:                                   # every other variant is finite there
        ok = plic.plic_solve(*dev(V0, nx, ny, nz), method=m, fast=f).cpu().numpy()
        assert np.max(np.abs(ok - (V0 - 0.5))) <= 2e-7, (m, f)
    px, py, pz = gen.paper_normals(4096, seed=22)
    E = plic.plic_roundtrip_error(*dev(px, py, pz), 64, method="kawano").cpu().numpy()
    assert np.isnan(E[0]) and np.isnan(E.astype(np.float64).mean())
    # (b) on normals whose smallest component is not small it is the same solution as the others
    #     ("apart from floating-point errors ... identical results"); the literal
    #     a2, a1, a0 arithmetic loses digits as m1 -> 0, hence the restriction and the looser bound
    V0, nx, ny, nz = gen.random_sphere(1 << 18, seed=23)
    keep = np.minimum(np.minimum(np.abs(nx), np.abs(ny)), np.abs(nz)) > 0.1
    V0, nx, ny, nz = V0[keep], nx[keep], ny[keep], nz[keep]
    ref = oracle.solve(V0, nx, ny, nz)
    got = plic.plic_solve(*dev(V0, nx, ny, nz), method="kawano").cpu().numpy()
    assert np.all(np.isfinite(got))
    assert np.max(np.abs(got.astype(np.float64) - ref)) <= 1e-4
    assert np.median(np.abs(got.astype(np.float64) - ref)) <= 2e-6


# ------------------------------------------------------------------------------------------
# adversarial normal / volume distributions (none of BASELINE.json's configs, all in the domain)
# ------------------------------------------------------------------------------------------
def test_adversarial_distributions(plic):
    rng = np.random.Generator(np.random.Philox(key=51))
    N = 1 << 19

    def unit(g):
        return g / np.linalg.norm(g, axis=1)[:, None]

    sets = {}
    g = rng.standard_normal((N, 3)); g[:, 0] *= 10.0 ** rng.uniform(-12, 0, N)
    sets["tiny n1"] = (unit(g), rng.random(N))
    g = rng.standard_normal((N, 3)); g[:, 0] *= 10.0 ** rng.uniform(-8, 0, N); g[:, 1] *= 10.0 ** rng.uniform(-8, 0, N)
    sets["tiny n1, n2"] = (unit(g), rng.random(N))
    g = np.abs(rng.standard_normal((N, 3))); g[:, 1] = g[:, 0] * (1 + rng.uniform(-1e-6, 1e-6, N))
    sets["n1 ~ n2"] = (unit(g), rng.random(N))
    g = np.ones((N, 3)) + rng.uniform(-1e-5, 1e-5, (N, 3))
    sets["n1 ~ n2 ~ n3"] = (unit(g), rng.random(N))
    third = N // 3
    sets["V0 near 0, 1, 1/2"] = (unit(rng.standard_normal((N, 3))), np.concatenate([
        10.0 ** rng.uniform(-12, -2, third), 1 - 10.0 ** rng.uniform(-7, -2, third),
        0.5 + rng.uniform(-1e-5, 1e-5, N - 2 * third)]))
    for name, (n, V) in sets.items():
        n = n[:, rng.permutation(3)] * rng.choice([-1.0, 1.0], (N, 3))
        V0 = V.astype(np.float32)
        nx, ny, nz = [np.ascontiguousarray(n[:, i].astype(np.float32)) for i in range(3)]
        ref = oracle.solve(V0, nx, ny, nz)
        for method, fast in VARIANTS:
            check_solve(plic, V0, nx, ny, nz, method, fast, ref=ref, what="%s / %s" % (name, method))
        d0 = (ref * rng.uniform(0.0, 1.0, N)).astype(np.float32)
        got = plic.plic_volume(*dev(d0, nx, ny, nz)).cpu().numpy().astype(np.float64)
        assert np.max(np.abs(got - oracle.volume(d0, nx, ny, nz))) <= TOL_VOL, name
