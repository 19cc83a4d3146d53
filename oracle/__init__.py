"""ctypes binding of the CPU oracle (oracle/oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of bench.py.  Nothing under
``paper_2107_05395_b200/`` imports this package and this package imports nothing from it.

All routines are fp64 and take / return numpy arrays.  The pentadiagonal routines use the
paper's diagonal names: a = 2nd sub-diagonal, b = sub-diagonal, c = main,
d = super-diagonal, e = 2nd super-diagonal.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

_lib = None


def sanitized() -> bool:
    """ORACLE_SANITIZE=1: build and load the oracle with AddressSanitizer + UndefinedBehaviorSanitizer (tests run the
    pin suite once that way, in a child process that preloads libasan; see tests/test_oracle_sanitized.py)."""
    return os.environ.get("ORACLE_SANITIZE", "") not in ("", "0")


def build(force: bool = False) -> str:
    """Compile oracle.c with gcc (-O2, FMA contraction off, OpenMP over systems)."""
    lib = os.path.join(_HERE, "liboracle_san.so") if sanitized() else _LIB
    if force or not os.path.exists(lib) or os.path.getmtime(lib) < os.path.getmtime(_SRC):
        tmp = lib + f".tmp{os.getpid()}"
        opt = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-fno-omit-frame-pointer"] \
            if sanitized() else ["-O2"]
        cmd = ["gcc", "-std=c99"] + opt + ["-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
                                           "-fvisibility=hidden", "-Wall", "-Wextra", "-o", tmp, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, lib)
    return lib


_dp = ctypes.POINTER(ctypes.c_double)
_ll = ctypes.c_longlong


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.orc_tri_factor.argtypes = [ctypes.c_int, _dp, _dp, _dp]
        lib.orc_tri_factor.restype = ctypes.c_int
        lib.orc_tri_solve.argtypes = [ctypes.c_int, _dp, _dp, _dp, _dp]
        lib.orc_tri_solve.restype = None
        for name in ("orc_penta_factor", "orc_penta_factor_general"):
            fn = getattr(lib, name)
            fn.argtypes = [ctypes.c_int, _dp, _dp, _dp, _dp, _dp]
            fn.restype = ctypes.c_int
        lib.orc_penta_solve.argtypes = [ctypes.c_int, _dp, _dp, _dp, _dp, _dp, _dp]
        lib.orc_penta_solve.restype = None
        lib.orc_ch_rhs.argtypes = [ctypes.c_int, _dp, ctypes.c_double, _dp]
        lib.orc_ch_rhs.restype = None
        lib.orc_tri_solve_interleaved.argtypes = [ctypes.c_int, _dp, _dp, _dp, _dp, _ll, _ll, _ll,
                                                  _ll, ctypes.c_int, ctypes.c_int]
        lib.orc_tri_solve_interleaved.restype = ctypes.c_int
        lib.orc_penta_solve_interleaved.argtypes = [ctypes.c_int, _dp, _dp, _dp, _dp, _dp, _dp, _ll,
                                                    _ll, _ll, _ll, ctypes.c_int, ctypes.c_int]
        lib.orc_penta_solve_interleaved.restype = ctypes.c_int
        lib.orc_ch_step_interleaved.argtypes = [ctypes.c_int, _dp, _dp, _dp, _dp, _dp, _dp, _ll,
                                                _ll, _ll, _ll, ctypes.c_double, ctypes.c_int,
                                                ctypes.c_int]
        lib.orc_ch_step_interleaved.restype = ctypes.c_int
        lib.orc_tri_periodic_factor.argtypes = [ctypes.c_int, _dp, _dp, _dp, _dp, _dp, _dp]
        lib.orc_tri_periodic_factor.restype = ctypes.c_int
        lib.orc_tri_periodic_solve.argtypes = [ctypes.c_int, _dp, _dp, _dp, _dp, ctypes.c_double,
                                               ctypes.c_double, _dp]
        lib.orc_tri_periodic_solve.restype = None
        lib.orc_tri_periodic_solve_interleaved.argtypes = [ctypes.c_int, _dp, _dp, _dp, _dp,
                                                           ctypes.c_double, ctypes.c_double, _dp, _ll,
                                                           _ll, _ll, _ll, ctypes.c_int, ctypes.c_int]
        lib.orc_tri_periodic_solve_interleaved.restype = ctypes.c_int
        lib.orc_penta_periodic_factor.argtypes = [ctypes.c_int, _dp, _dp, _dp, _dp, _dp, _dp, _dp, _dp]
        lib.orc_penta_periodic_factor.restype = ctypes.c_int
        lib.orc_penta_periodic_solve.argtypes = [ctypes.c_int] + [_dp] * 9
        lib.orc_penta_periodic_solve.restype = None
        lib.orc_ch_rhs_periodic.argtypes = [ctypes.c_int, _dp, ctypes.c_double, _dp]
        lib.orc_ch_rhs_periodic.restype = None
        lib.orc_penta_periodic_interleaved.argtypes = [ctypes.c_int] + [_dp] * 9 + [_ll, _ll, _ll, _ll, ctypes.c_int,
                                                                                    ctypes.c_double, ctypes.c_int, ctypes.c_int]
        lib.orc_penta_periodic_interleaved.restype = ctypes.c_int
        lib.orc_lbar_interleaved.argtypes = [ctypes.c_int, _dp, _ll]
        lib.orc_lbar_interleaved.restype = ctypes.c_double
        lib.orc_tri_explicit.argtypes = [ctypes.c_int, _dp, ctypes.c_double, ctypes.c_double, ctypes.c_double,
                                         ctypes.c_int, _dp]
        lib.orc_tri_explicit.restype = None
        lib.orc_tri_cn_step_interleaved.argtypes = [ctypes.c_int, _dp, _dp, _dp, _dp, ctypes.c_double, ctypes.c_double,
                                                    ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_double, _dp,
                                                    _ll, _ll, _ll, _ll, ctypes.c_int, ctypes.c_int]
        lib.orc_tri_cn_step_interleaved.restype = ctypes.c_int
        lib.orc_penta_explicit.argtypes = [ctypes.c_int, _dp, _dp, ctypes.c_int, _dp]
        lib.orc_penta_explicit.restype = None
        lib.orc_penta_cn_step_interleaved.argtypes = [ctypes.c_int] + [_dp] * 8 + [ctypes.c_int, _dp, _dp, _ll, _ll, _ll,
                                                                                   _ll, ctypes.c_int, ctypes.c_int]
        lib.orc_penta_cn_step_interleaved.restype = ctypes.c_int
        _lib = lib
    return _lib


def _p(x: np.ndarray):
    assert x.dtype == np.float64 and x.flags["C_CONTIGUOUS"]
    return x.ctypes.data_as(_dp)


def _f64(x) -> np.ndarray:
    return np.ascontiguousarray(np.array(x, dtype=np.float64, copy=True))


class FactorError(ArithmeticError):
    """Zero / non-finite pivot; ``row`` is the 1-based row (the paper has no pivoting)."""

    def __init__(self, row: int):
        super().__init__(f"zero or non-finite pivot at row {row}")
        self.row = row


@dataclass
class TriFactor:
    n: int
    a: np.ndarray   # untouched sub-diagonal
    bh: np.ndarray  # b^  (eq. 2)
    ch: np.ndarray  # c^  (eq. 1-2)


@dataclass
class PentaFactor:
    n: int
    eps: np.ndarray    # = a            (step 14)
    beta: np.ndarray   # overwrote b
    alpha: np.ndarray  # overwrote c
    gamma: np.ndarray  # overwrote d
    delta: np.ndarray  # overwrote e


def tri_factor(a, b, c) -> TriFactor:
    a, b, c = _f64(a), _f64(b), _f64(c)
    n = b.size
    assert a.size == n and c.size == n
    rc = _load().orc_tri_factor(n, _p(a), _p(b), _p(c))
    if rc:
        raise FactorError(rc)
    return TriFactor(n, a, b, c)


def tri_solve(fac: TriFactor, d) -> np.ndarray:
    """One contiguous system (length n); returns x."""
    x = _f64(d)
    assert x.shape == (fac.n,)
    _load().orc_tri_solve(fac.n, _p(fac.a), _p(fac.bh), _p(fac.ch), _p(x))
    return x


def penta_factor(a, b, c, d, e, general: bool = False) -> PentaFactor:
    a, b, c, d, e = (_f64(v) for v in (a, b, c, d, e))
    n = c.size
    assert all(v.size == n for v in (a, b, d, e))
    fn = _load().orc_penta_factor_general if general else _load().orc_penta_factor
    rc = fn(n, _p(a), _p(b), _p(c), _p(d), _p(e))
    if rc:
        raise FactorError(rc)
    return PentaFactor(n, a, b, c, d, e)


def penta_solve(fac: PentaFactor, f) -> np.ndarray:
    x = _f64(f)
    assert x.shape == (fac.n,)
    _load().orc_penta_solve(fac.n, _p(fac.eps), _p(fac.beta), _p(fac.alpha), _p(fac.gamma),
                            _p(fac.delta), _p(x))
    return x


def ch_rhs(c, alpha: float) -> np.ndarray:
    c = _f64(c)
    f = np.empty_like(c)
    _load().orc_ch_rhs(c.size, _p(c), float(alpha), _p(f))
    return f


def _subset(M, subset):
    jlo, jhi, jstride = (0, M, 1) if subset is None else subset
    assert 0 <= jlo <= jhi <= M and jstride >= 1
    return jlo, jhi, jstride


def tri_solve_interleaved(fac: TriFactor, rhs: np.ndarray, nsteps: int = 1, subset=None,
                          nthreads: int = 0) -> int:
    """In place on ``rhs`` of shape (n, M) (element i of system j at rhs[i, j]).
    ``subset=(jlo, jhi, jstride)`` restricts the systems touched.  Returns threads used."""
    assert rhs.ndim == 2 and rhs.shape[0] == fac.n
    M = rhs.shape[1]
    jlo, jhi, js = _subset(M, subset)
    return _load().orc_tri_solve_interleaved(fac.n, _p(fac.a), _p(fac.bh), _p(fac.ch), _p(rhs), M,
                                             jlo, jhi, js, nsteps, nthreads)


def penta_solve_interleaved(fac: PentaFactor, rhs: np.ndarray, nsteps: int = 1, subset=None,
                            nthreads: int = 0) -> int:
    assert rhs.ndim == 2 and rhs.shape[0] == fac.n
    M = rhs.shape[1]
    jlo, jhi, js = _subset(M, subset)
    return _load().orc_penta_solve_interleaved(fac.n, _p(fac.eps), _p(fac.beta), _p(fac.alpha),
                                               _p(fac.gamma), _p(fac.delta), _p(rhs), M, jlo, jhi,
                                               js, nsteps, nthreads)


def ch_step_interleaved(fac: PentaFactor, c: np.ndarray, alpha: float, nsteps: int = 1,
                        subset=None, nthreads: int = 0) -> int:
    """Config-5 stepper: nsteps x [f = c + alpha*D2(c^3-c); c = (I+sigma*D4)^-1 f], in place."""
    assert c.ndim == 2 and c.shape[0] == fac.n
    M = c.shape[1]
    jlo, jhi, js = _subset(M, subset)
    return _load().orc_ch_step_interleaved(fac.n, _p(fac.eps), _p(fac.beta), _p(fac.alpha),
                                           _p(fac.gamma), _p(fac.delta), _p(c), M, jlo, jhi, js,
                                           float(alpha), nsteps, nthreads)


# ---- periodic tridiagonal (eq. 12-15) ---------------------------------------------

@dataclass
class TriPeriodicFactor:
    n: int
    a: np.ndarray   # sub-diagonal; a[0] was the corner entry (row 1, column N)
    bh: np.ndarray  # b^ of A' (eq. 13b)
    ch: np.ndarray  # c^ of A'
    z: np.ndarray   # A'^{-1} u (eq. 14)
    vN: float       # last entry of v (eq. 13a)
    den: float      # 1 + v.z (eq. 15)


def tri_periodic_factor(a, b, c) -> TriPeriodicFactor:
    """Cyclic tridiagonal matrix: row i is a[i] x[i-1] + b[i] x[i] + c[i] x[i+1] with indices mod n,
    i.e. a[0] multiplies x[n-1] and c[n-1] multiplies x[0]."""
    a, b, c = _f64(a), _f64(b), _f64(c)
    n = b.size
    assert a.size == n and c.size == n
    z = np.zeros(n)
    vN, den = ctypes.c_double(0.0), ctypes.c_double(0.0)
    rc = _load().orc_tri_periodic_factor(n, _p(a), _p(b), _p(c), _p(z), ctypes.byref(vN), ctypes.byref(den))
    if rc:
        raise FactorError(rc)
    return TriPeriodicFactor(n, a, b, c, z, vN.value, den.value)


def tri_periodic_solve(fac: TriPeriodicFactor, d) -> np.ndarray:
    x = _f64(d)
    assert x.shape == (fac.n,)
    _load().orc_tri_periodic_solve(fac.n, _p(fac.a), _p(fac.bh), _p(fac.ch), _p(fac.z), fac.vN, fac.den, _p(x))
    return x


def tri_periodic_solve_interleaved(fac: TriPeriodicFactor, rhs: np.ndarray, nsteps: int = 1, subset=None,
                                   nthreads: int = 0) -> int:
    assert rhs.ndim == 2 and rhs.shape[0] == fac.n
    M = rhs.shape[1]
    jlo, jhi, js = _subset(M, subset)
    return _load().orc_tri_periodic_solve_interleaved(fac.n, _p(fac.a), _p(fac.bh), _p(fac.ch), _p(fac.z),
                                                      fac.vN, fac.den, _p(rhs), M, jlo, jhi, js, nsteps, nthreads)


# ---- periodic pentadiagonal (eq. 26a; Woodbury, C-31) and periodic CH step ------

@dataclass
class PentaPeriodicFactor:
    n: int
    eps: np.ndarray
    beta: np.ndarray
    alpha: np.ndarray
    gamma: np.ndarray
    delta: np.ndarray
    Z: np.ndarray    # (n, 4) = A'^{-1} U
    H: np.ndarray    # (4, 4) = (I + V^T Z)^{-1}
    w6: np.ndarray   # the six wrap-around entries


def penta_periodic_factor(a, b, c, d, e) -> PentaPeriodicFactor:
    """Cyclic pentadiagonal matrix, paper naming: row i is a[i] x[i-2] + b[i] x[i-1] + c[i] x[i] +
    d[i] x[i+1] + e[i] x[i+2] with indices mod n."""
    a, b, c, d, e = (_f64(v) for v in (a, b, c, d, e))
    n = c.size
    assert all(v.size == n for v in (a, b, d, e))
    Z, H, w6 = np.zeros((n, 4)), np.zeros((4, 4)), np.zeros(6)
    rc = _load().orc_penta_periodic_factor(n, _p(a), _p(b), _p(c), _p(d), _p(e), _p(Z), _p(H), _p(w6))
    if rc:
        raise FactorError(rc)
    return PentaPeriodicFactor(n, a, b, c, d, e, Z, H, w6)


def penta_periodic_solve(fac: PentaPeriodicFactor, f) -> np.ndarray:
    x = _f64(f)
    assert x.shape == (fac.n,)
    _load().orc_penta_periodic_solve(fac.n, _p(fac.eps), _p(fac.beta), _p(fac.alpha), _p(fac.gamma), _p(fac.delta),
                                     _p(fac.Z), _p(fac.H), _p(fac.w6), _p(x))
    return x


def ch_rhs_periodic(c, alpha: float) -> np.ndarray:
    c = _f64(c)
    f = np.zeros_like(c)
    _load().orc_ch_rhs_periodic(c.size, _p(c), alpha, _p(f))
    return f


def _penta_periodic_interleaved(fac, buf, mode, alpha_x, nsteps, subset, nthreads):
    assert buf.ndim == 2 and buf.shape[0] == fac.n
    M = buf.shape[1]
    jlo, jhi, js = _subset(M, subset)
    return _load().orc_penta_periodic_interleaved(fac.n, _p(fac.eps), _p(fac.beta), _p(fac.alpha), _p(fac.gamma),
                                                  _p(fac.delta), _p(fac.Z), _p(fac.H), _p(fac.w6), _p(buf), M, jlo,
                                                  jhi, js, mode, alpha_x, nsteps, nthreads)


def penta_periodic_solve_interleaved(fac: PentaPeriodicFactor, rhs: np.ndarray, nsteps: int = 1, subset=None,
                                     nthreads: int = 0) -> int:
    return _penta_periodic_interleaved(fac, rhs, 0, 0.0, nsteps, subset, nthreads)


def ch_periodic_step_interleaved(fac: PentaPeriodicFactor, c: np.ndarray, alpha: float, nsteps: int = 1,
                                 subset=None, nthreads: int = 0) -> int:
    return _penta_periodic_interleaved(fac, c, 1, alpha, nsteps, subset, nthreads)


# ---- coarsening statistic (eq. 30) ---------------------------------------------------

def lbar_interleaved(c: np.ndarray) -> float:
    """Mean over the runs (columns) of 1 / (1 - <C^2>), <C^2> = mean over the rows of C^2."""
    assert c.ndim == 2 and c.dtype == np.float64 and c.flags.c_contiguous
    return float(_load().orc_lbar_interleaved(c.shape[0], _p(c), c.shape[1]))


def ch_steps_with_lbar(fac, c: np.ndarray, alpha: float, nsteps: int, periodic: bool = True) -> np.ndarray:
    """Advance ``c`` in place ``nsteps`` steps, returning lbar after every step (eq. 30 "at every time-step")."""
    out = np.zeros(nsteps)
    for s in range(nsteps):
        if periodic:
            ch_periodic_step_interleaved(fac, c, alpha, nsteps=1)
        else:
            ch_step_interleaved(fac, c, alpha, nsteps=1)
        out[s] = lbar_interleaved(c)
    return out


# ---- Crank-Nicolson diffusion step (eq. 9-11) -----------------------------------------

def tri_explicit(c, xa: float, xb: float, xc: float, periodic: bool) -> np.ndarray:
    c = _f64(c)
    f = np.zeros_like(c)
    _load().orc_tri_explicit(c.size, _p(c), xa, xb, xc, int(periodic), _p(f))
    return f


def tri_cn_step_interleaved(fac, u: np.ndarray, xa: float, xb: float, xc: float, nsteps: int = 1, subset=None,
                            nthreads: int = 0) -> int:
    """``fac``: TriFactor (truncated) or TriPeriodicFactor (periodic).  In place on ``u`` (n, M)."""
    assert u.ndim == 2 and u.shape[0] == fac.n
    M = u.shape[1]
    jlo, jhi, js = _subset(M, subset)
    per = isinstance(fac, TriPeriodicFactor)
    z = fac.z if per else np.zeros(1)
    return _load().orc_tri_cn_step_interleaved(fac.n, _p(fac.a), _p(fac.bh), _p(fac.ch), _p(z),
                                               fac.vN if per else 0.0, fac.den if per else 1.0, int(per), xa, xb, xc,
                                               _p(u), M, jlo, jhi, js, nsteps, nthreads)


# ---- Crank-Nicolson hyperdiffusion step (eq. 17-19) -----------------------------------

def penta_explicit(c, x5, periodic: bool) -> np.ndarray:
    c, x5 = _f64(c), _f64(x5)
    assert x5.size == 5
    f = np.zeros_like(c)
    _load().orc_penta_explicit(c.size, _p(c), _p(x5), int(periodic), _p(f))
    return f


def penta_cn_step_interleaved(fac, u: np.ndarray, x5, nsteps: int = 1, subset=None, nthreads: int = 0) -> int:
    """``fac``: PentaFactor (truncated) or PentaPeriodicFactor (periodic).  In place on ``u`` (n, M)."""
    assert u.ndim == 2 and u.shape[0] == fac.n
    x5 = _f64(x5)
    assert x5.size == 5
    M = u.shape[1]
    jlo, jhi, js = _subset(M, subset)
    per = isinstance(fac, PentaPeriodicFactor)
    Z = fac.Z if per else np.zeros(4)
    H = fac.H if per else np.zeros(16)
    w6 = fac.w6 if per else np.zeros(6)
    return _load().orc_penta_cn_step_interleaved(fac.n, _p(fac.eps), _p(fac.beta), _p(fac.alpha), _p(fac.gamma),
                                                 _p(fac.delta), _p(Z), _p(H), _p(w6), int(per), _p(x5), _p(u), M,
                                                 jlo, jhi, js, nsteps, nthreads)
