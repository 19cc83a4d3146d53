"""Seeded synthetic inputs shared by the tests, bench.py and smoke().

This module holds NONE of the method's arithmetic (no factor, no sweep, no stencil): only the
counter-based random number generator and the recipes that turn BASELINE.json's configs into
LHS diagonals and right-hand sides.  It is the one module both the CPU oracle's tests and the
CUDA path's tests draw from.

Generator: value(seed, tag, j, i) = 2*u - 1 in [-1, 1), u = (z >> 11) * 2^-53,
    z = mix(mix(mix(seed + tag*G) + j) + i),  mix = the SplitMix64 finaliser,
keyed on (system j, row i) and not on i*batch+j, so a system's data does not depend on the batch
size and any subset of systems can be regenerated on its own.  Integer arithmetic and the
int -> double conversion are exact, so the numpy code here and the CUDA kernel in gen.cu produce
bit-identical arrays (tests/test_inputs.py).
"""
from __future__ import annotations

import ctypes
import math
import os
import subprocess

import numpy as np

_G = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)

TAG_RHS = 1        # uniform right-hand sides / initial fields
TAG_MODE_K = 2     # config 2: mode numbers
TAG_MODE_A = 3     # config 2: mode amplitudes


def _mix(z: np.ndarray) -> np.ndarray:
    z = z.astype(np.uint64, copy=True)
    z ^= z >> np.uint64(30)
    z *= _M1
    z ^= z >> np.uint64(27)
    z *= _M2
    z ^= z >> np.uint64(31)
    return z


def raw_bits(seed: int, tag: int, j, i) -> np.ndarray:
    """64 random bits for every (j, i) pair (broadcasting)."""
    with np.errstate(over="ignore"):
        s0 = _mix(np.asarray([(int(seed) + int(tag) * int(_G)) & 0xFFFFFFFFFFFFFFFF], dtype=np.uint64))
        s1 = _mix(s0 + np.asarray(j, dtype=np.uint64))
        return _mix(s1 + np.asarray(i, dtype=np.uint64))


def uniform_pm1(seed: int, tag: int, j, i) -> np.ndarray:
    """value(seed, tag, j, i) in [-1, 1), float64."""
    z = raw_bits(seed, tag, j, i)
    return (z >> np.uint64(11)).astype(np.float64) * (2.0 * 2.0 ** -53) - 1.0


def uniform_rhs(n: int, batch: int, seed: int = 0, scale: float = 1.0, dtype=np.float64,
                systems=None, tag: int = TAG_RHS) -> np.ndarray:
    """Interleaved array (n, batch) [element i of system j at [i, j]] of scale*value(seed, j, i).
    ``systems``: optional 1-D array of system indices j to generate instead of range(batch)."""
    j = np.arange(batch, dtype=np.uint64) if systems is None else np.asarray(systems, dtype=np.uint64)
    i = np.arange(n, dtype=np.uint64)
    out = uniform_pm1(seed, tag, j[None, :], i[:, None])
    if scale != 1.0:
        out = out * scale
    return np.ascontiguousarray(out.astype(dtype))


# ---- LHS recipes (BASELINE.json configs) -------------------------------------------------------

def tri_lhs(n: int, r: float = 0.5):
    """Configs 1, 2, 4: sub = super = -r, diag = 1 + 2r, truncated (a, b, c of btps.h)."""
    return np.full(n, -r), np.full(n, 1.0 + 2.0 * r), np.full(n, -r)


def penta_lhs(n: int, r: float = 0.5):
    """Configs 3, 4: I + r*[1,-4,6,-4,1] truncated at both ends (e, a, d, c, f of btps.h)."""
    return (np.full(n, r), np.full(n, -4.0 * r), np.full(n, 1.0 + 6.0 * r), np.full(n, -4.0 * r),
            np.full(n, r))


def ch_params(n: int = 256, g: float = 0.01, length: float = 2.0 * math.pi, dt: float = 5e-5):
    """Config 5: sigma = g*dt/dx^4 (LHS = I + sigma*D4), alpha = dt/dx^2, dx = L/n."""
    dx = length / n
    return g * dt / dx ** 4, dt / dx ** 2


def ch_lhs(n: int = 256, **kw):
    sigma, _ = ch_params(n, **kw)
    return penta_lhs(n, sigma)


def sine_modes_u0(n: int, batch: int, seed: int = 0, systems=None, nmodes: int = 4, kmax: int = 16):
    """Config 2 initial data: u_i = sum_m A_m sin(k_m pi x_i), x_i = i/(n+1), i = 1..n;
    k_m = 1 + (bits mod kmax), A_m = value(seed, TAG_MODE_A, j, m).
    Returns (u0 (n, batch) float64, k (nmodes, batch) int64, A (nmodes, batch) float64)."""
    j = np.arange(batch, dtype=np.uint64) if systems is None else np.asarray(systems, dtype=np.uint64)
    m = np.arange(nmodes, dtype=np.uint64)
    k = (raw_bits(seed, TAG_MODE_K, j[None, :], m[:, None]) % np.uint64(kmax)).astype(np.int64) + 1
    A = uniform_pm1(seed, TAG_MODE_A, j[None, :], m[:, None])
    x = np.arange(1, n + 1, dtype=np.float64) / (n + 1)
    u0 = np.zeros((n, j.size))
    for mm in range(nmodes):
        u0 += A[mm][None, :] * np.sin(np.pi * k[mm][None, :].astype(np.float64) * x[:, None])
    return np.ascontiguousarray(u0), k, A


# ---- device-side generator (same integers, CUDA) -----------------------------------------------

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gen.cu")
_LIB = os.path.join(_HERE, "libbtps_inputs.so")
_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        nvcc = "/usr/local/cuda/bin/nvcc" if os.path.exists("/usr/local/cuda/bin/nvcc") else "nvcc"
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-shared",
                        "-Xcompiler", "-fPIC", "-o", tmp, _SRC], check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.btps_inputs_fill_uniform.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int64,
                                                 ctypes.c_int64, ctypes.c_uint64, ctypes.c_uint64,
                                                 ctypes.c_double, ctypes.c_void_p]
        lib.btps_inputs_fill_uniform.restype = ctypes.c_int
        _lib = lib
    return _lib


def fill_uniform_device(t, n: int, seed: int = 0, scale: float = 1.0, tag: int = TAG_RHS, j0: int = 0,
                        stream=None):
    """Fill the CUDA tensor ``t`` (n*batch float64 or float32, interleaved) with
    scale*value(seed, tag, j0 + j, i), bit-identical to ``uniform_rhs``."""
    import torch
    assert t.is_cuda and t.is_contiguous() and t.numel() % n == 0
    elem = t.element_size()
    assert elem in (4, 8)
    st = torch.cuda.current_stream().cuda_stream if stream is None else int(stream)
    rc = _load().btps_inputs_fill_uniform(t.data_ptr(), elem, n, t.numel() // n, j0, seed, tag, scale, st)
    if rc != 0:
        raise RuntimeError(f"btps_inputs_fill_uniform failed with CUDA error {rc}")
    return t
