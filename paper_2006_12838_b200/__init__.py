"""paper_2006_12838_b200 -- Python binding of libplic (include/plic.h): argument marshalling only.

Every step of the PLIC path (mirror/sort, volume reduction, case selection, the per-case
solve, sign restore; eq. (1)-(8), (11), (25), (26)) runs in the CUDA kernels of
``csrc/``.  This module loads ``libplic.so`` with ctypes, passes raw device (or host)
pointers, sizes and the CUDA stream handle, and turns error codes into exceptions.  PyTorch
appears only as the owner of device memory and streams.  There is no CPU fallback: if the
shared library is missing it is built with nvcc, and if that fails the import raises.

    plic_solve(V0, nx, ny, nz, out=None, method="analytic", fast=False, stream=None) -> d0
    plic_volume(d0, nx, ny, nz, out=None, stream=None) -> V0
    plic_solve_host / plic_volume_host      same maps for host arrays (numpy or CPU tensors)
    plic_solve_h / plic_volume_h            the same maps on float16 tensors (fp32 arithmetic, 10 B/cell)
    plic_solve_f64                          plic_solve on float64 tensors in fp64 arithmetic (40 B/cell)
    plic_roundtrip_error(nx, ny, nz, L, out=None, method="analytic", fast=False) -> E
                                            the paper's benchmark loop, eq. (31)-(33)
    plic_sphere_solve(V0, out=None, fast=False) -> d0, plic_sphere_volume(d0, out=None) -> V0
                                            the plane-sphere intersection of sect. 3
    plic_curvature(phi, out=None, work=None) -> kappa
                                            curvature from a lattice of fill levels, sect. 4
    plic_curvature_static(phi, out=None) -> kappa
                                            the same without scratch from the caller (built-in list,
                                            lattices up to CURVATURE_STATIC_MAX_POINTS interior cells)
"""
from __future__ import annotations

import ctypes
import os

from . import build as _build

__all__ = ["METHODS", "FAST", "BLANK", "KAWANO", "method_id", "plic_solve", "plic_volume",
           "plic_solve_h", "plic_volume_h", "plic_solve_f64",
           "plic_roundtrip_error", "plic_sphere_solve", "plic_sphere_volume", "plic_curvature",
           "plic_curvature_static", "CURVATURE_STATIC_MAX_POINTS",
           "plic_solve_host",
           "plic_volume_host", "plic_host_release", "plic_method_name", "plic_error_string",
           "plic_version", "plic_launch_config", "plic_pipe_probe", "PROBES", "plic_launch_count", "PlicError", "lib",
           "LIB_PATH"]

METHODS = {"analytic": 0, "sz": 1, "newton": 2, "nested": 3}
KAWANO = 4              # Listing 3 (Kawano's SZ translation), precise only; see include/plic.h
FAST = 0x100
BLANK = 0x40            # the blank run of eq. (33): d0 = V0 - 1/2 (plic_roundtrip_error, plic_solve, plic_solve_h)
CURVATURE_STATIC_MAX_POINTS = (1 << 22) - 1     # PLIC_CURVATURE_STATIC_MAX_POINTS of include/plic.h
LIB_PATH = _build.LIB


class PlicError(RuntimeError):
    def __init__(self, code: int, what: str):
        super().__init__("%s failed: %s (code %d)" % (what, plic_error_string(code), code))
        self.code = code


def _load() -> ctypes.CDLL:
    path = _build.build()          # no-op when libplic.so is newer than its sources
    lib_ = ctypes.CDLL(path)
    fp = ctypes.c_void_p
    i64 = ctypes.c_int64
    ip = ctypes.POINTER(ctypes.c_int)
    lib_.plic_solve.argtypes = [fp, fp, fp, fp, fp, i64, ctypes.c_int, ctypes.c_void_p]
    lib_.plic_solve.restype = ctypes.c_int
    lib_.plic_volume.argtypes = [fp, fp, fp, fp, fp, i64, ctypes.c_void_p]
    lib_.plic_volume.restype = ctypes.c_int
    lib_.plic_solve_h.argtypes = [fp, fp, fp, fp, fp, fp, i64, ctypes.c_int, ctypes.c_void_p]
    lib_.plic_solve_h.restype = ctypes.c_int
    lib_.plic_volume_h.argtypes = [fp, fp, fp, fp, fp, fp, i64, ctypes.c_void_p]
    lib_.plic_volume_h.restype = ctypes.c_int
    lib_.plic_solve_f64.argtypes = [fp, fp, fp, fp, fp, i64, ctypes.c_int, ctypes.c_void_p]
    lib_.plic_solve_f64.restype = ctypes.c_int
    lib_.plic_roundtrip_error.argtypes = [fp, fp, fp, fp, i64, ctypes.c_int, ctypes.c_int,
                                          ctypes.c_void_p]
    lib_.plic_roundtrip_error.restype = ctypes.c_int
    lib_.plic_sphere_solve.argtypes = [fp, fp, i64, ctypes.c_int, ctypes.c_void_p]
    lib_.plic_sphere_solve.restype = ctypes.c_int
    lib_.plic_sphere_volume.argtypes = [fp, fp, i64, ctypes.c_void_p]
    lib_.plic_sphere_volume.restype = ctypes.c_int
    lib_.plic_curvature.argtypes = [fp, fp, ctypes.c_int, ctypes.c_int, ctypes.c_int, fp, i64,
                                    ctypes.c_void_p]
    lib_.plic_curvature.restype = ctypes.c_int
    lib_.plic_curvature_static.argtypes = [fp, fp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_void_p]
    lib_.plic_curvature_static.restype = ctypes.c_int
    lib_.plic_solve_host.argtypes = [fp, fp, fp, fp, fp, i64, ctypes.c_int]
    lib_.plic_solve_host.restype = ctypes.c_int
    lib_.plic_volume_host.argtypes = [fp, fp, fp, fp, fp, i64]
    lib_.plic_volume_host.restype = ctypes.c_int
    lib_.plic_host_release.argtypes = []
    lib_.plic_host_release.restype = None
    lib_.plic_method_name.argtypes = [ctypes.c_int]
    lib_.plic_method_name.restype = ctypes.c_char_p
    lib_.plic_error_string.argtypes = [ctypes.c_int]
    lib_.plic_error_string.restype = ctypes.c_char_p
    lib_.plic_version.argtypes = []
    lib_.plic_version.restype = ctypes.c_int
    lib_.plic_launch_config.argtypes = [ctypes.c_int, i64, ip, ip, ip]
    lib_.plic_launch_config.restype = ctypes.c_int
    lib_.plic_pipe_probe.argtypes = [ctypes.c_int, ctypes.c_int, fp, ctypes.POINTER(i64), ctypes.c_void_p]
    lib_.plic_pipe_probe.restype = ctypes.c_int
    lib_.plic_launch_count.argtypes = []
    lib_.plic_launch_count.restype = i64
    return lib_


lib = _load()


def method_id(method, fast: bool = False) -> int:
    """'analytic' | 'sz' | 'newton' | 'nested' (optionally with a '-fast' suffix) or an int id."""
    if isinstance(method, str):
        name = method
        if name.endswith("-fast"):
            name, fast = name[:-5], True
        if name == "blank":
            return BLANK
        if name == "kawano":
            if fast:
                raise ValueError("the kawano method has no fast form")
            return KAWANO
        if name not in METHODS:
            raise ValueError("unknown PLIC method %r" % (method,))
        mid = METHODS[name]
    else:
        mid = int(method)
    return mid | (FAST if fast else 0)


def plic_method_name(method: int):
    s = lib.plic_method_name(int(method))
    return s.decode() if s is not None else None


def plic_error_string(code: int) -> str:
    return lib.plic_error_string(int(code)).decode()


def plic_version() -> int:
    return int(lib.plic_version())


def plic_launch_count() -> int:
    return int(lib.plic_launch_count())


def plic_launch_config(method, N: int, fast: bool = False):
    """(grid, block, cells_per_thread) of plic_solve (method id/name) or plic_volume (method=-1)."""
    g, b, c = ctypes.c_int(), ctypes.c_int(), ctypes.c_int()
    mid = -1 if method == -1 else method_id(method, fast)
    rc = lib.plic_launch_config(mid, int(N), ctypes.byref(g), ctypes.byref(b), ctypes.byref(c))
    if rc != 0:
        raise PlicError(rc, "plic_launch_config")
    return g.value, b.value, c.value


PROBES = {"ffma": 0, "ffma2": 1, "mufu": 2, "fmnmx": 3, "lop3": 4, "nested_step": 5, "ffma+lop3": 6,
          "ffma2+lop3": 7, "mufu+4ffma": 8, "ffma+fmnmx": 9, "fsetp+fsel": 10, "nested_step_scalar": 11,
          "nested_step_hybrid": 12, "fadd": 13, "fmul": 14, "fadd2": 15, "2ffma+lop3+fadd": 16, "dfma": 17}


def plic_pipe_probe(pipe, trips: int, sink, stream=None) -> int:
    """Enqueues one instruction-rate probe launch (include/plic.h); returns the number of
    warp-instructions of the probed kind that launch executes.  `sink`: float32 CUDA tensor, >= 256."""
    n = i64_out = ctypes.c_int64(0)
    pid = PROBES[pipe] if isinstance(pipe, str) else int(pipe)
    rc = lib.plic_pipe_probe(pid, int(trips), sink.data_ptr(), ctypes.byref(i64_out),
                             _stream_handle(stream, sink.device))
    if rc != 0:
        raise PlicError(rc, "plic_pipe_probe")
    return int(n.value)


def plic_host_release() -> None:
    lib.plic_host_release()


# ------------------------------------------------------------------------------------------
# device-pointer API (torch CUDA tensors)
# ------------------------------------------------------------------------------------------
def _device_args(first, nx, ny, nz, out, dtype=None):
    import torch
    dtype = torch.float32 if dtype is None else dtype
    N = first.numel()
    for t in (first, nx, ny, nz):
        if not (t.is_cuda and t.dtype == dtype and t.dim() == 1 and t.is_contiguous()
                and t.numel() == N and t.device == first.device):
            raise ValueError("inputs must be contiguous 1-D %s CUDA tensors of one length "
                             "on one device" % (dtype,))
    if out is None:
        out = torch.empty_like(first)
    elif not (out.is_cuda and out.dtype == dtype and out.is_contiguous()
              and out.numel() == N and out.device == first.device):
        raise ValueError("out must be a contiguous %s CUDA tensor of the inputs' length" % (dtype,))
    return N, out


def _aux_ptr(aux, N, device):
    """Optional float32 side output of the binary16 maps: data pointer or None."""
    import torch
    if aux is None:
        return None
    if not (aux.is_cuda and aux.dtype == torch.float32 and aux.is_contiguous() and aux.numel() == N
            and aux.device == device):
        raise ValueError("out_f32 must be a contiguous float32 CUDA tensor of the inputs' length")
    return aux.data_ptr()


def _stream_handle(stream, device):
    import torch
    if stream is None:
        stream = torch.cuda.current_stream(device)
    return ctypes.c_void_p(int(stream.cuda_stream) if hasattr(stream, "cuda_stream") else int(stream))


def plic_solve(V0, nx, ny, nz, out=None, method="analytic", fast: bool = False, stream=None):
    """d0 = d0(V0, n) per cell (eq. (1)) on the tensors' device; returns `out`."""
    import torch
    N, out = _device_args(V0, nx, ny, nz, out)
    with torch.cuda.device(V0.device):
        rc = lib.plic_solve(V0.data_ptr(), nx.data_ptr(), ny.data_ptr(), nz.data_ptr(),
                            out.data_ptr(), N, method_id(method, fast),
                            _stream_handle(stream, V0.device))
    if rc != 0:
        raise PlicError(rc, "plic_solve")
    return out


def plic_volume(d0, nx, ny, nz, out=None, stream=None):
    """V0 = V0(d0, n) per cell (eq. (6), (7), (11)) on the tensors' device; returns `out`."""
    import torch
    N, out = _device_args(d0, nx, ny, nz, out)
    with torch.cuda.device(d0.device):
        rc = lib.plic_volume(d0.data_ptr(), nx.data_ptr(), ny.data_ptr(), nz.data_ptr(),
                             out.data_ptr(), N, _stream_handle(stream, d0.device))
    if rc != 0:
        raise PlicError(rc, "plic_volume")
    return out


def plic_solve_h(V0, nx, ny, nz, out=None, out_f32=None, method="analytic", fast: bool = False, stream=None):
    """plic_solve on float16 tensors (binary16 storage, fp32 arithmetic); `out_f32`, if given, also
    receives the float32 result before it is rounded to float16.  Returns `out` (float16)."""
    import torch
    N, out = _device_args(V0, nx, ny, nz, out, torch.float16)
    with torch.cuda.device(V0.device):
        rc = lib.plic_solve_h(V0.data_ptr(), nx.data_ptr(), ny.data_ptr(), nz.data_ptr(), out.data_ptr(),
                              _aux_ptr(out_f32, N, V0.device), N, method_id(method, fast),
                              _stream_handle(stream, V0.device))
    if rc != 0:
        raise PlicError(rc, "plic_solve_h")
    return out


def plic_volume_h(d0, nx, ny, nz, out=None, out_f32=None, stream=None):
    """plic_volume on float16 tensors (binary16 storage, fp32 arithmetic).  Returns `out` (float16)."""
    import torch
    N, out = _device_args(d0, nx, ny, nz, out, torch.float16)
    with torch.cuda.device(d0.device):
        rc = lib.plic_volume_h(d0.data_ptr(), nx.data_ptr(), ny.data_ptr(), nz.data_ptr(), out.data_ptr(),
                               _aux_ptr(out_f32, N, d0.device), N, _stream_handle(stream, d0.device))
    if rc != 0:
        raise PlicError(rc, "plic_volume_h")
    return out


def plic_solve_f64(V0, nx, ny, nz, out=None, method="analytic", stream=None):
    """plic_solve on float64 tensors in fp64 arithmetic (precise methods only).  Returns `out`."""
    import torch
    N, out = _device_args(V0, nx, ny, nz, out, torch.float64)
    with torch.cuda.device(V0.device):
        rc = lib.plic_solve_f64(V0.data_ptr(), nx.data_ptr(), ny.data_ptr(), nz.data_ptr(), out.data_ptr(),
                                N, method_id(method, False), _stream_handle(stream, V0.device))
    if rc != 0:
        raise PlicError(rc, "plic_solve_f64")
    return out


def plic_roundtrip_error(nx, ny, nz, L: int, out=None, method="analytic", fast: bool = False,
                         stream=None):
    """E[i] = mean over L equally spaced V0 of |plic_volume(plic_solve(V0, n_i), n_i) - V0|
    (eq. (31)); method "blank" = eq. (33).  Returns `out`."""
    import torch
    N, out = _device_args(nx, nx, ny, nz, out)
    with torch.cuda.device(nx.device):
        rc = lib.plic_roundtrip_error(nx.data_ptr(), ny.data_ptr(), nz.data_ptr(), out.data_ptr(),
                                      N, int(L), method_id(method, fast),
                                      _stream_handle(stream, nx.device))
    if rc != 0:
        raise PlicError(rc, "plic_roundtrip_error")
    return out


def plic_sphere_solve(V0, out=None, fast: bool = False, stream=None):
    """d0 of the plane cutting the volume V0 off the unit-volume sphere (eq. (38)); returns `out`."""
    import torch
    N, out = _device_args(V0, V0, V0, V0, out)
    with torch.cuda.device(V0.device):
        rc = lib.plic_sphere_solve(V0.data_ptr(), out.data_ptr(), N, FAST if fast else 0,
                                   _stream_handle(stream, V0.device))
    if rc != 0:
        raise PlicError(rc, "plic_sphere_solve")
    return out


def plic_sphere_volume(d0, out=None, stream=None):
    """V0 cut off the unit-volume sphere by the plane at offset d0 (eq. (37)); returns `out`."""
    import torch
    N, out = _device_args(d0, d0, d0, d0, out)
    with torch.cuda.device(d0.device):
        rc = lib.plic_sphere_volume(d0.data_ptr(), out.data_ptr(), N,
                                    _stream_handle(stream, d0.device))
    if rc != 0:
        raise PlicError(rc, "plic_sphere_volume")
    return out


def plic_curvature(phi, out=None, work=None, stream=None):
    """kappa (eq. (63)) on a lattice of fill levels phi[z, y, x] (3-D contiguous float32 CUDA
    tensor); `work` is an int32 CUDA tensor of scratch (default: 1 + phi.numel() entries).
    Returns `out`; work[0] then holds the number of interface points."""
    import torch
    if not (phi.is_cuda and phi.dtype == torch.float32 and phi.dim() == 3 and phi.is_contiguous()):
        raise ValueError("phi must be a contiguous 3-D float32 CUDA tensor [nz, ny, nx]")
    if out is None:
        out = torch.empty_like(phi)
    elif not (out.is_cuda and out.dtype == torch.float32 and out.is_contiguous()
              and out.shape == phi.shape and out.device == phi.device):
        raise ValueError("out must be a contiguous float32 CUDA tensor of phi's shape")
    if work is None:
        work = torch.empty(1 + phi.numel(), dtype=torch.int32, device=phi.device)
    elif not (work.is_cuda and work.dtype == torch.int32 and work.is_contiguous()
              and work.device == phi.device):
        raise ValueError("work must be a contiguous int32 CUDA tensor")
    nz, ny, nx = phi.shape
    with torch.cuda.device(phi.device):
        rc = lib.plic_curvature(phi.data_ptr(), out.data_ptr(), nx, ny, nz, work.data_ptr(),
                                work.numel(), _stream_handle(stream, phi.device))
    if rc != 0:
        raise PlicError(rc, "plic_curvature")
    return out


def plic_curvature_static(phi, out=None, stream=None):
    """plic_curvature for callers that cannot allocate device memory where they need curvature (a solver
    whose lattices already fill the GPU, an application with its own device-memory pool, a time-step
    loop that must not hit cudaMalloc's device-wide synchronisation): the interface list is a fixed
    16 MiB array inside libplic instead of a `work` tensor.  Pass `out` (e.g. a buffer of the solver)
    and the call allocates nothing at all; with out=None only the result tensor comes from torch.

    Accepts lattices with at most CURVATURE_STATIC_MAX_POINTS cells off the border ((nx-2)(ny-2)(nz-2),
    e.g. 163^3); larger ones raise PlicError (code -6) before any GPU work -- use plic_curvature there.
    The first call on a device looks up the array's address: make it at start-up, outside stream
    capture.  All calls on one GPU share the list, so calls that may overlap on the GPU (two streams
    with no event between them) race; calls on one stream are fine.  kappa is bitwise that of
    plic_curvature.  Returns `out`."""
    import torch
    if not (phi.is_cuda and phi.dtype == torch.float32 and phi.dim() == 3 and phi.is_contiguous()):
        raise ValueError("phi must be a contiguous 3-D float32 CUDA tensor [nz, ny, nx]")
    if out is None:
        out = torch.empty_like(phi)
    elif not (out.is_cuda and out.dtype == torch.float32 and out.is_contiguous()
              and out.shape == phi.shape and out.device == phi.device):
        raise ValueError("out must be a contiguous float32 CUDA tensor of phi's shape")
    nz, ny, nx = phi.shape
    with torch.cuda.device(phi.device):
        rc = lib.plic_curvature_static(phi.data_ptr(), out.data_ptr(), nx, ny, nz,
                                       _stream_handle(stream, phi.device))
    if rc != 0:
        raise PlicError(rc, "plic_curvature_static")
    return out


# ------------------------------------------------------------------------------------------
# host-pointer API (numpy arrays or CPU torch tensors, pinned or pageable)
# ------------------------------------------------------------------------------------------
def _host_ptr(a, N=None):
    import numpy as np
    if hasattr(a, "data_ptr"):                       # CPU torch tensor
        import torch
        if a.is_cuda or a.dtype != torch.float32 or not a.is_contiguous() or a.dim() != 1:
            raise ValueError("host arrays must be contiguous 1-D float32 CPU tensors")
        n, p = a.numel(), a.data_ptr()
    else:
        if not (isinstance(a, np.ndarray) and a.dtype == np.float32 and a.ndim == 1
                and a.flags.c_contiguous):
            raise ValueError("host arrays must be contiguous 1-D float32 numpy arrays")
        n, p = a.shape[0], a.ctypes.data
    if N is not None and n != N:
        raise ValueError("host arrays must have one length")
    return n, p


def _host_out(first, out):
    import numpy as np
    if out is not None:
        return out
    if hasattr(first, "data_ptr"):
        import torch
        return torch.empty_like(first)
    return np.empty_like(first)


def plic_solve_host(V0, nx, ny, nz, out=None, method="analytic", fast: bool = False):
    """plic_solve for host arrays: chunked H2D / kernel / D2H pipeline inside libplic."""
    N, p0 = _host_ptr(V0)
    ptrs = [p0] + [_host_ptr(a, N)[1] for a in (nx, ny, nz)]
    out = _host_out(V0, out)
    ptrs.append(_host_ptr(out, N)[1])
    rc = lib.plic_solve_host(*ptrs, N, method_id(method, fast))
    if rc != 0:
        raise PlicError(rc, "plic_solve_host")
    return out


def plic_volume_host(d0, nx, ny, nz, out=None):
    """plic_volume for host arrays."""
    N, p0 = _host_ptr(d0)
    ptrs = [p0] + [_host_ptr(a, N)[1] for a in (nx, ny, nz)]
    out = _host_out(d0, out)
    ptrs.append(_host_ptr(out, N)[1])
    rc = lib.plic_volume_host(*ptrs, N)
    if rc != 0:
        raise PlicError(rc, "plic_volume_host")
    return out
