"""Builds paper_2006_12838_b200/libplic.so from csrc/ with nvcc for sm_100a (in-tree).

    python -m paper_2006_12838_b200.build [--force] [--verbose]

The .so is git-ignored but travels to the GPU box with the gpurun snapshot.  The CUDA runtime
is linked statically, so the library depends only on the driver (libcuda via the runtime's
dlopen) and libstdc++.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libplic.so")
SOURCES = [os.path.join(CSRC, "plic_kernels.cu")]
DEPENDS = SOURCES + [os.path.join(CSRC, "plic_methods.cuh"), os.path.join(CSRC, "plic_math.cuh"),
                     os.path.join(CSRC, "plic_packed.cuh"), os.path.join(CSRC, "plic_curvature.cuh"),
                     os.path.join(CSRC, "plic_probe.cuh"), os.path.join(CSRC, "plic_storage.cuh"),
                     os.path.join(CSRC, "plic_f64.cuh"), os.path.join(CSRC, "plic_curvature_static.cuh"),
                     os.path.join(ROOT, "include", "plic.h")]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC", "-cudart", "static"]


def find_nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libplic cannot be built (there is no CPU fallback)")


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(p) > t for p in DEPENDS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not is_stale():
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [find_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + SOURCES
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose:
        sys.stderr.write(res.stderr)
    if res.returncode != 0:
        if os.path.exists(tmp):
            os.remove(tmp)
        raise RuntimeError("nvcc failed:\n%s\n%s" % (" ".join(cmd), res.stderr))
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
