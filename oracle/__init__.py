"""fp64 CPU oracle for the PLIC plane-cube problem -- TEST INFRASTRUCTURE, NOT PRODUCT.

Thin ctypes loader around ``oracle/plic_oracle.c`` (plain C, fp64, gcc).  Only
``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from
``paper_2006_12838_b200`` and shares no code with the CUDA path; the arithmetic
lives entirely in the C file, whose header cites the paper passages it follows
(eq. (2)-(7), (11) of /root/reference/PAPER.md) and lists the readings taken.

    volume(d0, nx, ny, nz) -> V0      forward map, eq. (11)+(6)+(7)
    solve(V0, nx, ny, nz)  -> d0      bisection of the forward map on [-S/2, S/2]
    case(d0, nx, ny, nz)   -> 1..5    intersection case of eq. (11)

``oracle.stratified`` (``stratified.c``) generates the case-stratified workload of BASELINE.json
configs[2], which by its definition needs the case classifier and the forward map above; it is an
input generator for tests and for bench.py's divergence leg, not part of the oracle's arithmetic.

Sub-modules (numpy fp64, same rules): ``oracle.sphere`` -- the plane-sphere problem of sect. 3
(eq. (37) and its inverse by bisection); ``oracle.curvature`` -- the curvature calculation of
sect. 4 / appendix B (PY normal, PLIC point neighbourhood, paraboloid fit, eq. (63)).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "plic_oracle.c")
_SRC_STRAT = os.path.join(_HERE, "stratified.c")    # configs[2] workload generator (inputs, not the oracle)
_LIB = os.path.join(_HERE, "libplic_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile plic_oracle.c with gcc (-O2, no fast-math, OpenMP) next to the source."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC),
                                                                         os.path.getmtime(_SRC_STRAT)):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        cmd = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
               "-o", tmp, _SRC, _SRC_STRAT, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        fp = ctypes.POINTER(ctypes.c_float)
        ip = ctypes.POINTER(ctypes.c_int32)
        i64, i32, dbl = ctypes.c_int64, ctypes.c_int, ctypes.c_double
        lib.oracle_plic_volume.argtypes = [dbl] * 4
        lib.oracle_plic_volume.restype = dbl
        lib.oracle_plic_solve.argtypes = [dbl] * 4
        lib.oracle_plic_solve.restype = dbl
        lib.oracle_plic_case.argtypes = [dbl] * 4
        lib.oracle_plic_case.restype = i32
        lib.oracle_plic_volume_batch.argtypes = [dp, dp, dp, dp, dp, i64, i32]
        lib.oracle_plic_solve_batch.argtypes = [dp, dp, dp, dp, dp, i64, i32]
        lib.oracle_plic_case_batch.argtypes = [dp, dp, dp, dp, ip, i64, i32]
        lib.oracle_plic_volume_batch_f32.argtypes = [fp, fp, fp, fp, dp, i64, i32]
        lib.oracle_plic_solve_batch_f32.argtypes = [fp, fp, fp, fp, dp, i64, i32]
        lib.oracle_max_threads.restype = i32
        for f in (lib.oracle_plic_volume_batch, lib.oracle_plic_solve_batch,
                  lib.oracle_plic_case_batch, lib.oracle_plic_volume_batch_f32,
                  lib.oracle_plic_solve_batch_f32):
            f.restype = None
        _lib = lib
    return _lib


def _prep(*arrays):
    """Broadcast to a common 1-D shape; keep an all-fp32 set as fp32, else promote to fp64."""
    arrs = [np.asarray(a) for a in arrays]
    shape = np.broadcast_shapes(*[a.shape for a in arrs])
    all_f32 = all(a.dtype == np.float32 for a in arrs)
    dt = np.float32 if all_f32 else np.float64
    out = [np.ascontiguousarray(np.broadcast_to(a.astype(dt, copy=False), shape)).ravel()
           for a in arrs]
    return out, shape, all_f32


def _ptr(a, ctype):
    return a.ctypes.data_as(ctypes.POINTER(ctype))


def max_threads() -> int:
    return int(_load().oracle_max_threads())


def volume(d0, nx, ny, nz, threads: int = 0) -> np.ndarray:
    """V0(d0, n) in fp64.  Inputs fp32 (promoted exactly) or fp64; broadcastable."""
    lib = _load()
    (a, b, c, d), shape, f32 = _prep(d0, nx, ny, nz)
    out = np.empty(a.shape[0], dtype=np.float64)
    if f32:
        lib.oracle_plic_volume_batch_f32(*[_ptr(x, ctypes.c_float) for x in (a, b, c, d)],
                                         _ptr(out, ctypes.c_double), a.shape[0], threads)
    else:
        lib.oracle_plic_volume_batch(*[_ptr(x, ctypes.c_double) for x in (a, b, c, d)],
                                     _ptr(out, ctypes.c_double), a.shape[0], threads)
    return out.reshape(shape)


def solve(V0, nx, ny, nz, threads: int = 0) -> np.ndarray:
    """d0(V0, n) in fp64 by bisection.  Inputs fp32 (promoted exactly) or fp64."""
    lib = _load()
    (a, b, c, d), shape, f32 = _prep(V0, nx, ny, nz)
    out = np.empty(a.shape[0], dtype=np.float64)
    if f32:
        lib.oracle_plic_solve_batch_f32(*[_ptr(x, ctypes.c_float) for x in (a, b, c, d)],
                                        _ptr(out, ctypes.c_double), a.shape[0], threads)
    else:
        lib.oracle_plic_solve_batch(*[_ptr(x, ctypes.c_double) for x in (a, b, c, d)],
                                    _ptr(out, ctypes.c_double), a.shape[0], threads)
    return out.reshape(shape)


def case(d0, nx, ny, nz, threads: int = 0) -> np.ndarray:
    """Intersection case 1..5 of eq. (11) for the plane (d0, n); 0 for the zero normal."""
    lib = _load()
    arrs = [np.asarray(a, dtype=np.float64) for a in (d0, nx, ny, nz)]
    shape = np.broadcast_shapes(*[a.shape for a in arrs])
    a, b, c, d = [np.ascontiguousarray(np.broadcast_to(x, shape)).ravel() for x in arrs]
    out = np.empty(a.shape[0], dtype=np.int32)
    lib.oracle_plic_case_batch(*[_ptr(x, ctypes.c_double) for x in (a, b, c, d)],
                               _ptr(out, ctypes.c_int32), a.shape[0], threads)
    return out.reshape(shape)
