"""CPU-side checks of the C-ABI boundary: libplic.so builds, loads, and exports every
function include/plic.h declares; argument validation that returns before any CUDA call;
method-id marshalling of the Python binding.  No compute happens here (there is no GPU and
no CPU fallback)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def plic():
    import paper_2006_12838_b200 as p
    return p


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "plic.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(plic_[a-z_]+)\s*\(", src)))


def test_header_declares_the_boundary():
    names = _declared_functions()
    for must in ("plic_solve", "plic_volume", "plic_roundtrip_error", "plic_sphere_solve",
                 "plic_sphere_volume", "plic_curvature", "plic_solve_host", "plic_volume_host",
                 "plic_method_name", "plic_version", "plic_launch_count"):
        assert must in names


def test_library_exports_every_declared_symbol(plic):
    assert os.path.exists(plic.LIB_PATH)
    raw = ctypes.CDLL(plic.LIB_PATH)
    for name in _declared_functions():
        assert hasattr(raw, name), name


def test_header_compiles_as_plain_c(tmp_path):
    import subprocess
    c = tmp_path / "t.c"
    c.write_text('#include "plic.h"\nint main(void){return PLIC_NUM_METHODS==4?0:1;}\n')
    subprocess.run(["gcc", "-std=c11", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"),
                    "-c", str(c), "-o", str(tmp_path / "t.o")], check=True)


def test_version_and_names(plic):
    assert plic.plic_version() == 106
    assert [plic.plic_method_name(i) for i in range(4)] == ["analytic", "sz", "newton", "nested"]
    assert plic.plic_method_name(2 | plic.FAST) == "newton-fast"
    assert plic.plic_method_name(4) == "kawano" and plic.plic_method_name(4 | plic.FAST) is None
    assert plic.plic_method_name(5) is None and plic.plic_method_name(-1) is None
    assert plic.plic_method_name(plic.BLANK) == "blank"
    assert plic.plic_error_string(0) == "ok"
    for code in (-1, -2, -3, -4, -5, -6):
        assert plic.plic_error_string(code) not in ("ok", "unknown error code")


def test_method_id_marshalling(plic):
    assert plic.method_id("analytic") == 0
    assert plic.method_id("sz", fast=True) == 0x101
    assert plic.method_id("nested-fast") == 0x103
    assert plic.method_id(2) == 2
    assert plic.method_id("blank") == 0x40
    assert plic.method_id("kawano") == 4
    with pytest.raises(ValueError):
        plic.method_id("kawano-fast")
    with pytest.raises(ValueError):
        plic.method_id("applic")


def test_argument_validation_needs_no_device(plic):
    lib = plic.lib
    buf = (ctypes.c_float * 8)()
    p = ctypes.cast(buf, ctypes.c_void_p)
    # N == 0: successful no-op, even with null pointers
    assert lib.plic_solve(None, None, None, None, None, 0, 0, None) == 0
    assert lib.plic_volume(None, None, None, None, None, 0, None) == 0
    assert lib.plic_solve_host(None, None, None, None, None, 0, 0) == 0
    # N < 0
    assert lib.plic_solve(p, p, p, p, p, -1, 0, None) == -2
    assert lib.plic_volume(p, p, p, p, p, -5, None) == -2
    # null pointer with N > 0
    assert lib.plic_solve(p, None, p, p, p, 4, 0, None) == -1
    assert lib.plic_solve_host(p, p, p, p, None, 4, 0) == -1
    # unknown method
    assert lib.plic_solve(p, p, p, p, p, 4, 7, None) == -3
    assert lib.plic_solve(p, p, p, p, p, 4, 0x204, None) == -3
    assert lib.plic_solve(p, p, p, p, p, 4, 0x104, None) == -3               # kawano has no fast form
    assert lib.plic_solve_host(p, p, p, p, p, 4, -1) == -3
    # storage variants: same validation order; fp64 has the four precise methods only
    assert lib.plic_solve_h(None, None, None, None, None, None, 0, 0, None) == 0
    assert lib.plic_solve_h(p, p, p, p, p, None, -1, 0, None) == -2
    assert lib.plic_solve_h(p, p, None, p, p, None, 4, 0x100, None) == -1
    assert lib.plic_solve_h(p, p, p, p, p, None, 4, 0x204, None) == -3
    assert lib.plic_solve_h(ctypes.c_void_p(p.value + 1), p, p, p, p, None, 4, 0, None) == -5
    assert lib.plic_solve_h(p, p, p, p, p, ctypes.c_void_p(p.value + 2), 4, 0, None) == -5
    assert lib.plic_volume_h(None, None, None, None, None, None, 0, None) == 0
    assert lib.plic_volume_h(p, p, p, None, p, None, 4, None) == -1
    assert lib.plic_solve_f64(None, None, None, None, None, 0, 0, None) == 0
    assert lib.plic_solve_f64(p, p, p, p, p, -1, 0, None) == -2
    assert lib.plic_solve_f64(p, p, p, p, None, 2, 3, None) == -1
    assert lib.plic_solve_f64(p, p, p, p, p, 2, 0x100, None) == -3             # no fast form in fp64
    assert lib.plic_solve_f64(p, p, p, p, p, 2, 4, None) == -3                 # no kawano
    assert lib.plic_solve_f64(p, p, p, p, p, 2, 0x40, None) == -3              # no blank
    assert lib.plic_solve_f64(ctypes.c_void_p(p.value + 4), p, p, p, p, 2, 0, None) == -5
    # plic_roundtrip_error: sizes, method, null
    assert lib.plic_roundtrip_error(None, None, None, None, 0, 256, 0, None) == 0
    assert lib.plic_roundtrip_error(p, p, p, p, 4, 1, 0, None) == -2
    assert lib.plic_roundtrip_error(p, p, p, p, -4, 256, 0, None) == -2
    assert lib.plic_roundtrip_error(p, p, p, p, 4, 256, 9, None) == -3
    assert lib.plic_roundtrip_error(p, p, None, p, 4, 256, 0x40, None) == -1
    assert lib.plic_solve(p, p, p, p, p, 4, 0x140, None) == -3              # blank has no fast form
    assert lib.plic_solve(p, None, p, p, p, 4, 0x40, None) == -1            # blank is a plic_solve method (stream ceiling)
    # plane-sphere entry points
    assert lib.plic_sphere_solve(None, None, 0, 0, None) == 0
    assert lib.plic_sphere_solve(p, p, -1, 0, None) == -2
    assert lib.plic_sphere_solve(p, None, 4, 0, None) == -1
    assert lib.plic_sphere_solve(p, p, 4, 1, None) == -3
    assert lib.plic_sphere_volume(None, p, 4, None) == -1
    assert lib.plic_sphere_volume(ctypes.c_void_p(p.value + 2), p, 1, None) == -5
    # plic_curvature
    assert lib.plic_curvature(None, None, 0, 5, 5, None, 0, None) == 0
    assert lib.plic_curvature(p, p, -1, 5, 5, p, 8, None) == -2
    assert lib.plic_curvature(p, p, 2048, 2048, 2048, p, 8, None) == -2      # >= 2^31 cells
    assert lib.plic_curvature(p, p, 2, 2, 2, None, 8, None) == -1
    assert lib.plic_curvature(p, p, 2, 2, 2, p, 1, None) == -2
    # misaligned (not a multiple of 4 bytes)
    q = ctypes.c_void_p(p.value + 2)
    assert lib.plic_solve(q, p, p, p, p, 1, 0, None) == -5
    assert plic.plic_launch_count() == 0


def test_binding_rejects_wrong_tensors(plic):
    import numpy as np
    import torch
    a = torch.zeros(4)
    with pytest.raises(ValueError):
        plic.plic_solve(a, a, a, a)                       # CPU tensors on the device API
    with pytest.raises(ValueError):
        plic.plic_solve_host(np.zeros(4), np.zeros(4, np.float32), np.zeros(4, np.float32),
                             np.zeros(4, np.float32))     # float64 array
    with pytest.raises(ValueError):
        plic.plic_solve_host(np.zeros(4, np.float32), np.zeros(3, np.float32),
                             np.zeros(4, np.float32), np.zeros(4, np.float32))


def test_no_oracle_in_product_path():
    """The product (package, include/) never imports or links the oracle."""
    pkg = os.path.join(ROOT, "paper_2006_12838_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, f
                assert "plic_oracle" not in txt, f
