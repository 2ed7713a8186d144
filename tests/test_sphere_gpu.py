"""GPU parity of plic_sphere_solve / plic_sphere_volume (sect. 3) against oracle/sphere.py,
element by element through the C ABI.  Tolerances: |d0 - ref| <= 2e-6 and |V0 - ref| <= 1e-6
(a handful of fp32 operations on quantities <= 1)."""
import numpy as np
import pytest
import torch

from oracle import sphere

pytestmark = pytest.mark.gpu

TOL_D0 = 2e-6
TOL_V0 = 1e-6
R = sphere.R


@pytest.fixture(scope="module")
def plic():
    import paper_2006_12838_b200 as p
    return p


def volumes(n, seed):
    """V0 ~ U[0,1) plus a log-spaced approach to both ends and the exact edge values."""
    rng = np.random.Generator(np.random.Philox(key=seed))
    v = rng.random(n)
    edge = np.concatenate([10.0 ** np.linspace(-30, -1, 300), 1.0 - 10.0 ** np.linspace(-7.2, -1, 300),
                           [0.0, 0.5, 1.0, 1e-7, 1 - 1e-7, 5.0 / 32.0, 27.0 / 32.0]])
    return np.concatenate([v, edge]).astype(np.float32)


@pytest.mark.parametrize("fast", [False, True], ids=["precise", "fast"])
def test_sphere_solve_parity(plic, fast):
    V0 = volumes(1 << 20, 31)
    ref = sphere.sphere_solve(V0)
    before = plic.plic_launch_count()
    got = plic.plic_sphere_solve(torch.from_numpy(V0).cuda(), fast=fast).cpu().numpy()
    assert plic.plic_launch_count() > before
    assert got.dtype == np.float32 and np.all(np.isfinite(got))
    err = np.abs(got.astype(np.float64) - ref)
    i = int(np.argmax(err))
    assert err.max() <= TOL_D0, (err.max(), V0[i], got[i], ref[i])
    assert np.all(np.abs(got) <= np.float32(R) * (1 + 1e-6))
    # forward residual through the oracle; the cut-disc area is <= pi r^2 = 1.21
    res = np.abs(sphere.sphere_volume(got) - V0.astype(np.float64))
    assert res.max() <= 3e-6
    # exact values
    sel = {0.0: -R, 1.0: R, 0.5: 0.0, 5.0 / 32.0: -R / 2, 27.0 / 32.0: R / 2}
    for v, d in sel.items():
        j = np.where(V0 == np.float32(v))[0]
        assert len(j) and np.all(np.abs(got[j] - d) <= TOL_D0)


def test_sphere_volume_parity(plic):
    rng = np.random.Generator(np.random.Philox(key=32))
    d0 = np.concatenate([(rng.random(1 << 20) * 2 - 1) * R, [-R, R, 0.0, -R / 2, R / 2, -1.0, 1.0, 0.7],
                         -R + 10.0 ** np.linspace(-7, -1, 200), R - 10.0 ** np.linspace(-7, -1, 200)]).astype(np.float32)
    ref = sphere.sphere_volume(d0)
    got = plic.plic_sphere_volume(torch.from_numpy(d0).cuda()).cpu().numpy()
    assert np.all(np.isfinite(got)) and got.min() >= 0.0 and got.max() <= 1.0
    assert np.max(np.abs(got.astype(np.float64) - ref)) <= TOL_V0
    # small caps keep relative accuracy (cap form evaluated from the near pole)
    small = (ref > 0) & (ref < 1e-3)
    assert np.max(np.abs(got[small] / ref[small] - 1.0)) <= 1e-5


@pytest.mark.parametrize("fast", [False, True], ids=["precise", "fast"])
def test_sphere_ragged_misaligned_alias_empty(plic, fast):
    V0 = volumes(70001 - 607, 33)
    assert len(V0) == 70001
    ref = sphere.sphere_solve(V0)
    t = torch.from_numpy(V0).cuda()
    for N in (0, 1, 3, 4, 5, 255, 1027, 70001):
        out = plic.plic_sphere_solve(t[:N], fast=fast)
        assert out.shape == (N,)
        if N:
            assert np.max(np.abs(out.cpu().numpy().astype(np.float64) - ref[:N])) <= TOL_D0
    for off in (1, 2, 3):
        N = 4099
        out = torch.full((off + N + 5,), 7.0, device="cuda")
        plic.plic_sphere_solve(t[off:off + N], out=out[off:off + N], fast=fast)
        got = out.cpu().numpy()
        assert np.all(got[:off] == 7.0) and np.all(got[off + N:] == 7.0)
        assert np.max(np.abs(got[off:off + N].astype(np.float64) - ref[off:off + N])) <= TOL_D0
    # different alignment of input and output: scalar kernel, bitwise equal to the vector body
    a = plic.plic_sphere_solve(t, fast=fast)
    buf = torch.empty(70002, device="cuda")
    b = plic.plic_sphere_solve(t, out=buf[1:], fast=fast)
    assert torch.equal(a, b)
    c = t.clone()
    plic.plic_sphere_solve(c, out=c, fast=fast)                          # in place
    assert torch.equal(a, c)


def test_sphere_round_trip(plic):
    V0 = volumes(1 << 18, 34)
    t = torch.from_numpy(V0).cuda()
    back = plic.plic_sphere_volume(plic.plic_sphere_solve(t, fast=True)).cpu().numpy()
    assert np.max(np.abs(back.astype(np.float64) - V0)) <= 3e-6
