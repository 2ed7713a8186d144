"""plic_curvature_static: the curvature call for callers that cannot allocate device memory.

plic_curvature leaves its interface list (`work`) to the caller.  A flow solver whose lattices
already fill the GPU, an application that manages device memory through its own pool, or a time-step
loop that must stay clear of cudaMalloc's device-wide synchronisation cannot supply one, so
plic_curvature_static keeps the list in a fixed 16 MiB array inside libplic and limits the lattice
to PLIC_CURVATURE_STATIC_MAX_POINTS interior cells (include/plic.h).

What is checked here: its kappa equals the kappa of plic_curvature (same kernels, so bit for bit --
the bar tests/test_curvature_gpu.py sets for the aligned against the unaligned call) on two calls in a
row, where the second lattice has FEWER interface points than the first, so that entries the first
call left in the shared list would show up if the counter were not cleared; that a call allocates
no device memory; and that a lattice beyond the limit is refused with its own error code.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure in this
optional entry point must not hide the parity tests.  The GPU test passes alone in a fresh process
(the first call does the per-device set-up) and after the rest of the suite."""
import ctypes
import os
import sys

import numpy as np
import pytest

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def plic():
    import paper_2006_12838_b200 as p
    return p


def test_limit_is_checked_before_any_device_work(plic):
    """Needs no GPU: the size checks come first.  164^3 has 162^3 = 4 251 528 interior cells > the limit."""
    raw = ctypes.CDLL(plic.LIB_PATH)
    raw.plic_curvature_static.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_int,
                                          ctypes.c_int, ctypes.c_void_p]
    raw.plic_curvature_static.restype = ctypes.c_int
    fake = ctypes.c_void_p(256)                                   # never dereferenced
    assert plic.CURVATURE_STATIC_MAX_POINTS == 4194303
    assert 161 ** 3 <= plic.CURVATURE_STATIC_MAX_POINTS < 162 ** 3
    assert raw.plic_curvature_static(fake, fake, 164, 164, 164, None) == -6
    assert raw.plic_curvature_static(fake, fake, 256, 256, 256, None) == -6
    assert raw.plic_curvature_static(fake, fake, -1, 8, 8, None) == -2
    assert raw.plic_curvature_static(fake, fake, 2048, 2048, 2048, None) == -2      # >= 2^31 cells
    assert raw.plic_curvature_static(None, fake, 8, 8, 8, None) == -1
    msg = plic.plic_error_string(-6)
    assert "PLIC_CURVATURE_STATIC_MAX_POINTS" in msg and "plic_curvature" in msg


@pytest.mark.gpu
def test_static_matches_caller_scratch_path_on_two_calls_in_a_row(plic):
    import torch
    import lattices
    # call 1: a drop of radius 20 (about 7000 interface points); call 2: radius 7 in a lattice of
    # another shape whose x extent is not a multiple of 4 (about 900 points, scalar tail in the marker)
    cases = [lattices.sphere((56, 60, 64), (32.3, 29.6, 27.9), 20.0),
             lattices.sphere((30, 33, 37), (18.2, 16.4, 14.9), 7.0)]
    phis = [torch.from_numpy(np.ascontiguousarray(p)).cuda() for p in cases]
    refs, counts = [], []
    for t in phis:                                                # the existing path, scratch from torch
        work = torch.empty(1 + t.numel(), dtype=torch.int32, device="cuda")
        refs.append(plic.plic_curvature(t, work=work).clone())
        counts.append(int(work[0].item()))
    assert counts[0] > 4 * counts[1] > 400                        # the second list is much shorter
    outs = [torch.full_like(t, float("nan")) for t in phis]      # every cell must be written
    torch.cuda.synchronize()
    plic.plic_curvature_static(phis[0], out=outs[0])              # warm: per-device set-up happens here at the latest
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    launches = plic.plic_launch_count()
    for t, o in zip(phis, outs):                                  # two calls in a row on one stream
        o.fill_(float("nan"))
        plic.plic_curvature_static(t, out=o)
    torch.cuda.synchronize()
    assert plic.plic_launch_count() == launches + 6               # 3 kernels per call, as plic_curvature
    assert torch.cuda.mem_get_info()[0] == free_before             # free device memory unchanged: nothing allocated
    for t, o, r in zip(phis, outs, refs):
        assert torch.equal(o, r)                                  # bitwise (NaN anywhere would fail too)
        assert int((o != 0).sum().item()) > 0
    # and once more in the opposite order, the long list after the short one
    for i in (1, 0):
        outs[i].fill_(float("nan"))
        plic.plic_curvature_static(phis[i], out=outs[i])
    torch.cuda.synchronize()
    for o, r in zip(outs, refs):
        assert torch.equal(o, r)
    # a lattice beyond the limit is refused through the binding too, and kappa is left alone
    big = torch.zeros((164, 164, 164), dtype=torch.float32, device="cuda")
    out = torch.full_like(big, 7.0)
    with pytest.raises(plic.PlicError) as ei:
        plic.plic_curvature_static(big, out=out)
    assert ei.value.code == -6
    torch.cuda.synchronize()
    assert bool((out == 7.0).all().item())
    # the largest accepted cube
    ok = torch.zeros((163, 163, 163), dtype=torch.float32, device="cuda")
    ok[80, 80, 80] = 0.5
    k = plic.plic_curvature_static(ok)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(k).all().item())
