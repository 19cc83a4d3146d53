"""ctypes marshalling for include/btps.h.  No arithmetic of the method lives here."""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libbtps.so")

# every symbol include/btps.h declares (tests check the library exports each of them)
EXPORTS = [
    "tri_factor", "tri_factor_periodic", "tri_destroy", "penta_factor", "penta_factor_periodic", "penta_destroy",
    "tri_solve_batched", "tri_solve_batched_f32", "penta_solve_batched", "penta_solve_batched_f32",
    "tri_solve_batched_f32s", "penta_solve_batched_f32s",
    "tri_solve_steps", "penta_solve_steps", "ch_step_batched", "ch_step_batched_stat", "tri_cn_step_batched", "penta_cn_step_batched",
    "tri_solve_batched_host", "penta_solve_batched_host", "ch_step_batched_host", "tri_solve_batched_host_static",
    "btps_last_error", "btps_error_string", "btps_plan_info", "btps_tune", "btps_launch_count", "btps_kernel_tag",
    "btps_build_id",
]


class BtpsError(RuntimeError):
    def __init__(self, code: int, msg: str, row: int = 0):
        super().__init__(f"btps error {code}: {msg}" + (f" (row {row})" if row else ""))
        self.code = code
        self.row = row


def lib_path() -> str:
    return _LIB_PATH


def _load() -> ctypes.CDLL:
    if not os.path.exists(_LIB_PATH):
        raise ImportError(
            f"{_LIB_PATH} is missing: build it with `python -m paper_2107_05395_b200.build` "
            "(there is no CPU / PyTorch fallback for this library)")
    lib = ctypes.CDLL(_LIB_PATH)
    vp, dp, fp, i64, ci = ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.c_void_p, \
        ctypes.c_int64, ctypes.c_int
    lib.tri_factor.argtypes = [ci, dp, dp, dp]
    lib.tri_factor.restype = vp
    lib.tri_factor_periodic.argtypes = [ci, dp, dp, dp]
    lib.tri_factor_periodic.restype = vp
    lib.tri_destroy.argtypes = [vp]
    lib.tri_destroy.restype = None
    lib.penta_factor.argtypes = [ci, dp, dp, dp, dp, dp]
    lib.penta_factor.restype = vp
    lib.penta_factor_periodic.argtypes = [ci, dp, dp, dp, dp, dp]
    lib.penta_factor_periodic.restype = vp
    lib.penta_destroy.argtypes = [vp]
    lib.penta_destroy.restype = None
    for name in ("tri_solve_batched", "tri_solve_batched_f32", "penta_solve_batched",
                 "penta_solve_batched_f32", "tri_solve_batched_f32s", "penta_solve_batched_f32s"):
        fn = getattr(lib, name)
        fn.argtypes = [vp, vp, i64, vp]
        fn.restype = ci
    for name in ("tri_solve_steps", "penta_solve_steps"):
        fn = getattr(lib, name)
        fn.argtypes = [vp, vp, i64, ci, vp]
        fn.restype = ci
    lib.ch_step_batched.argtypes = [vp, vp, i64, ctypes.c_double, ci, vp]
    lib.ch_step_batched.restype = ci
    lib.tri_cn_step_batched.argtypes = [vp, vp, i64, ctypes.c_double, ctypes.c_double, ctypes.c_double, ci, vp]
    lib.tri_cn_step_batched.restype = ci
    lib.penta_cn_step_batched.argtypes = [vp, vp, i64, dp, ci, vp]
    lib.penta_cn_step_batched.restype = ci
    lib.ch_step_batched_stat.argtypes = [vp, vp, i64, ctypes.c_double, ci, vp, vp]
    lib.ch_step_batched_stat.restype = ci
    for name in ("tri_solve_batched_host", "penta_solve_batched_host"):
        fn = getattr(lib, name)
        fn.argtypes = [vp, vp, i64, ci]
        fn.restype = ci
    lib.ch_step_batched_host.argtypes = [vp, vp, i64, ctypes.c_double, ci]
    lib.ch_step_batched_host.restype = ci
    lib.tri_solve_batched_host_static.argtypes = [vp, vp, i64, ci, vp]
    lib.tri_solve_batched_host_static.restype = ci
    lib.btps_last_error.argtypes = [ctypes.POINTER(ci)]
    lib.btps_last_error.restype = ci
    lib.btps_error_string.argtypes = [ci]
    lib.btps_error_string.restype = ctypes.c_char_p
    lib.btps_plan_info.argtypes = [ci, vp, ci, ctypes.POINTER(ci)]
    lib.btps_plan_info.restype = ci
    lib.btps_tune.argtypes = [ctypes.c_char_p, ci]
    lib.btps_tune.restype = ci
    lib.btps_launch_count.argtypes = []
    lib.btps_launch_count.restype = i64
    lib.btps_kernel_tag.argtypes = [ci, vp, ci, i64, ci, ctypes.c_char_p, ci]
    lib.btps_kernel_tag.restype = ci
    lib.btps_build_id.argtypes = []
    lib.btps_build_id.restype = ctypes.c_char_p
    return lib


_lib = _load()


def _raise_last():
    row = ctypes.c_int(0)
    code = _lib.btps_last_error(ctypes.byref(row))
    raise BtpsError(code, _lib.btps_error_string(code).decode(), row.value)


def _check(rc: int):
    if rc != 0:
        _raise_last()


def _host64(x) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(x, dtype=np.float64))


def _dptr(x):
    return x.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


class _Handle:
    _destroy = None
    kind = -1

    def __init__(self, ptr: int, n: int):
        self.ptr = ptr
        self.n = n

    def close(self):
        if self.ptr:
            type(self)._destroy(self.ptr)
            self.ptr = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def plan(self, elem_bytes: int = 8) -> dict:
        return btps_plan_info(self, elem_bytes)


class TriHandle(_Handle):
    _destroy = staticmethod(lambda p: _lib.tri_destroy(p))
    kind = 0

    def cn_plan(self, elem_bytes: int = 8) -> dict:
        """Plan of the fused Crank-Nicolson step kernels of this handle (btps_plan_info kind 3)."""
        return btps_plan_info(self, elem_bytes, kind=3)


class PentaHandle(_Handle):
    _destroy = staticmethod(lambda p: _lib.penta_destroy(p))
    kind = 1

    def ch_plan(self, elem_bytes: int = 8) -> dict:
        """Plan of the fused Cahn-Hilliard step kernels of this handle (btps_plan_info kind 2)."""
        return btps_plan_info(self, elem_bytes, kind=2)

    def cn_plan(self, elem_bytes: int = 8) -> dict:
        """Plan of the fused Crank-Nicolson hyperdiffusion step kernels (btps_plan_info kind 4)."""
        return btps_plan_info(self, elem_bytes, kind=4)


def tri_factor(a, b, c) -> TriHandle:
    """btps.h tri_factor: host arrays a (sub), b (main), c (super), each length n."""
    a, b, c = _host64(a), _host64(b), _host64(c)
    n = b.size
    if a.size != n or c.size != n:
        raise ValueError("a, b, c must have the same length")
    ptr = _lib.tri_factor(n, _dptr(a), _dptr(b), _dptr(c))
    if not ptr:
        _raise_last()
    return TriHandle(ptr, n)


def tri_factor_periodic(a, b, c) -> TriHandle:
    """btps.h tri_factor_periodic: cyclic tridiagonal matrix (a[0] and c[n-1] are the corner entries);
    the handle is used with the same tri_solve_* calls."""
    a, b, c = _host64(a), _host64(b), _host64(c)
    n = b.size
    if a.size != n or c.size != n:
        raise ValueError("a, b, c must have the same length")
    ptr = _lib.tri_factor_periodic(n, _dptr(a), _dptr(b), _dptr(c))
    if not ptr:
        _raise_last()
    return TriHandle(ptr, n)


def penta_factor(e, a, d, c, f) -> PentaHandle:
    """btps.h penta_factor: host arrays e (2nd sub), a (sub), d (main), c (super), f (2nd super)."""
    e, a, d, c, f = (_host64(v) for v in (e, a, d, c, f))
    n = d.size
    if any(v.size != n for v in (e, a, c, f)):
        raise ValueError("e, a, d, c, f must have the same length")
    ptr = _lib.penta_factor(n, _dptr(e), _dptr(a), _dptr(d), _dptr(c), _dptr(f))
    if not ptr:
        _raise_last()
    return PentaHandle(ptr, n)


def penta_factor_periodic(e, a, d, c, f) -> PentaHandle:
    """btps.h penta_factor: host arrays e (2nd sub), a (sub), d (main), c (super), f (2nd super)."""
    e, a, d, c, f = (_host64(v) for v in (e, a, d, c, f))
    n = d.size
    if any(v.size != n for v in (e, a, c, f)):
        raise ValueError("e, a, d, c, f must have the same length")
    ptr = _lib.penta_factor_periodic(n, _dptr(e), _dptr(a), _dptr(d), _dptr(c), _dptr(f))
    if not ptr:
        _raise_last()
    return PentaHandle(ptr, n)


_torch = None
_raw_stream = None


def _torch_mod():
    """torch, imported on first use (callers hold device memory in torch tensors; nothing here computes with it)."""
    global _torch, _raw_stream
    if _torch is None:
        import torch
        _torch = torch
        # the current stream's raw handle without building a torch.cuda.Stream object (the object costs ~3 us per call)
        _raw_stream = getattr(torch._C, "_cuda_getCurrentRawStream", None)
    return _torch


def _dev_args(h: _Handle, t, elem_bytes: int):
    """t: a CUDA torch tensor holding n*batch elements (any shape, contiguous) -> (ptr, batch)."""
    torch = _torch or _torch_mod()
    if t.dtype is not (torch.float64 if elem_bytes == 8 else torch.float32):
        raise ValueError(f"expected a floating tensor with {elem_bytes}-byte elements")
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError("expected a contiguous CUDA tensor")
    size = t.numel()
    if size % h.n:
        raise ValueError("tensor size is not a multiple of n")
    return t.data_ptr(), size // h.n


def _stream(stream):
    if stream is None:
        torch = _torch or _torch_mod()
        if _raw_stream is not None:
            return _raw_stream(torch.cuda.current_device())
        return torch.cuda.current_stream().cuda_stream
    return int(stream)


def tri_solve_batched(h: TriHandle, rhs, stream=None):
    p, batch = _dev_args(h, rhs, 8)
    _check(_lib.tri_solve_batched(h.ptr, p, batch, _stream(stream)))


def tri_solve_batched_f32(h: TriHandle, rhs, stream=None):
    p, batch = _dev_args(h, rhs, 4)
    _check(_lib.tri_solve_batched_f32(h.ptr, p, batch, _stream(stream)))


def penta_solve_batched(h: PentaHandle, rhs, stream=None):
    p, batch = _dev_args(h, rhs, 8)
    _check(_lib.penta_solve_batched(h.ptr, p, batch, _stream(stream)))


def penta_solve_batched_f32(h: PentaHandle, rhs, stream=None):
    p, batch = _dev_args(h, rhs, 4)
    _check(_lib.penta_solve_batched_f32(h.ptr, p, batch, _stream(stream)))


def tri_solve_batched_f32s(h: TriHandle, rhs, stream=None):
    """btps.h tri_solve_batched_f32s: float32 tensor in HBM, fp64 arithmetic."""
    p, batch = _dev_args(h, rhs, 4)
    _check(_lib.tri_solve_batched_f32s(h.ptr, p, batch, _stream(stream)))


def penta_solve_batched_f32s(h: PentaHandle, rhs, stream=None):
    p, batch = _dev_args(h, rhs, 4)
    _check(_lib.penta_solve_batched_f32s(h.ptr, p, batch, _stream(stream)))


def tri_solve_steps(h: TriHandle, rhs, nsteps: int, stream=None):
    p, batch = _dev_args(h, rhs, 8)
    _check(_lib.tri_solve_steps(h.ptr, p, batch, int(nsteps), _stream(stream)))


def penta_solve_steps(h: PentaHandle, rhs, nsteps: int, stream=None):
    p, batch = _dev_args(h, rhs, 8)
    _check(_lib.penta_solve_steps(h.ptr, p, batch, int(nsteps), _stream(stream)))


def ch_step_batched(h: PentaHandle, c, alpha: float, nsteps: int = 1, stream=None):
    p, batch = _dev_args(h, c, 8)
    _check(_lib.ch_step_batched(h.ptr, p, batch, float(alpha), int(nsteps), _stream(stream)))


def tri_cn_step_batched(h: TriHandle, u, xa: float, xb: float, xc: float, nsteps: int = 1, stream=None):
    p, batch = _dev_args(h, u, 8)
    _check(_lib.tri_cn_step_batched(h.ptr, p, batch, float(xa), float(xb), float(xc), int(nsteps), _stream(stream)))


def penta_cn_step_batched(h: PentaHandle, u, x5, nsteps: int = 1, stream=None):
    p, batch = _dev_args(h, u, 8)
    x5 = _host64(x5)
    if x5.size != 5:
        raise ValueError("x5 must hold the five explicit stencil coefficients")
    _check(_lib.penta_cn_step_batched(h.ptr, p, batch, _dptr(x5), int(nsteps), _stream(stream)))


def ch_step_batched_stat(h: PentaHandle, c, alpha: float, nsteps: int, lbar, stream=None):
    """btps.h ch_step_batched_stat: ``lbar`` is a CUDA float64 tensor of nsteps elements (overwritten)."""
    p, batch = _dev_args(h, c, 8)
    if not (lbar.is_cuda and lbar.is_contiguous() and lbar.element_size() == 8 and lbar.numel() >= int(nsteps)):
        raise ValueError("lbar must be a contiguous CUDA float64 tensor with at least nsteps elements")
    _check(_lib.ch_step_batched_stat(h.ptr, p, batch, float(alpha), int(nsteps), lbar.data_ptr(), _stream(stream)))


def _host_args(h: _Handle, x):
    """x: a C-contiguous float64 host buffer (numpy array or CPU torch tensor) of n*batch values."""
    if hasattr(x, "data_ptr"):  # torch CPU tensor (possibly pinned)
        if x.is_cuda or not x.is_contiguous() or x.element_size() != 8:
            raise ValueError("expected a contiguous float64 CPU tensor")
        ptr, size = x.data_ptr(), x.numel()
    else:
        if x.dtype != np.float64 or not x.flags["C_CONTIGUOUS"]:
            raise ValueError("expected a C-contiguous float64 array")
        ptr, size = x.ctypes.data, x.size
    if size % h.n:
        raise ValueError("buffer size is not a multiple of n")
    return ptr, size // h.n


def tri_solve_batched_host(h: TriHandle, rhs, nsteps: int = 1):
    p, batch = _host_args(h, rhs)
    _check(_lib.tri_solve_batched_host(h.ptr, p, batch, int(nsteps)))


def penta_solve_batched_host(h: PentaHandle, rhs, nsteps: int = 1):
    p, batch = _host_args(h, rhs)
    _check(_lib.penta_solve_batched_host(h.ptr, p, batch, int(nsteps)))


def ch_step_batched_host(h: PentaHandle, c, alpha: float, nsteps: int = 1):
    p, batch = _host_args(h, c)
    _check(_lib.ch_step_batched_host(h.ptr, p, batch, float(alpha), int(nsteps)))


STATIC_SCRATCH_BYTES = 32 << 20  # btps.h BTPS_STATIC_SCRATCH_BYTES


def tri_solve_batched_host_static(h: TriHandle, rhs, nsteps: int = 1, stream=None):
    """btps.h tri_solve_batched_host_static: the host-buffer solve that allocates nothing (n*batch*8 <= 32 MiB)."""
    p, batch = _host_args(h, rhs)
    _check(_lib.tri_solve_batched_host_static(h.ptr, p, batch, int(nsteps), _stream(stream)))


def btps_last_error():
    row = ctypes.c_int(0)
    code = _lib.btps_last_error(ctypes.byref(row))
    return code, row.value, _lib.btps_error_string(code).decode()


_PLAN_KEYS = ("rows_per_thread", "partitions", "lanes", "systems_per_thread", "tiles_per_cta",
              "threads_per_cta", "smem_bytes", "table_bytes", "tma_prefetch", "warp_scan")


def btps_plan_info(h: _Handle, elem_bytes: int = 8, kind: int = None) -> dict:
    out = (ctypes.c_int * 10)()
    _check(_lib.btps_plan_info(h.kind if kind is None else kind, h.ptr, elem_bytes, out))
    return dict(zip(_PLAN_KEYS, list(out)))


def btps_tune(key: str, value: int):
    _check(_lib.btps_tune(key.encode(), int(value)))


def btps_launch_count() -> int:
    return int(_lib.btps_launch_count())


def btps_kernel_tag(h: _Handle, elem_bytes: int, batch: int, nsteps: int = 1, kind: int = None) -> str:
    """btps.h btps_kernel_tag: template arguments of the kernel such a call would launch (nothing is launched)."""
    buf = ctypes.create_string_buffer(96)
    _check(_lib.btps_kernel_tag(h.kind if kind is None else kind, h.ptr, elem_bytes, int(batch), int(nsteps), buf, 96))
    return buf.value.decode()


def btps_build_id() -> str:
    return _lib.btps_build_id().decode()
