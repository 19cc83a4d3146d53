"""Pins for the tridiagonal oracle (oracle/oracle.c: orc_tri_factor / orc_tri_solve).

Every expected value here comes from something other than the oracle: exact rational Gaussian
elimination, numpy's dense LAPACK solve, textbook closed forms.  No GPU needed.
"""
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle
from tests._exact import dense_from_bands, exact_solve, np_dense_from_bands, read_golden


def tri_bands(a, b, c):
    return {-1: a, 0: b, 1: c}


def toeplitz_tri(n, r):
    return np.full(n, -r), np.full(n, 1 + 2 * r), np.full(n, -r)


# --- worked example, exact rationals (tests/golden/tri_n4.txt) ---------------------------------

def test_worked_example_n4(golden_dir):
    g = read_golden(os.path.join(golden_dir, "tri_n4.txt"))
    n = 4
    # the fixture itself is pinned by exact elimination (independent of the oracle)
    A = dense_from_bands(n, tri_bands(g["a"], g["b"], g["c"]))
    assert exact_solve(A, g["d"]) == g["x"]
    fac = oracle.tri_factor([float(v) for v in g["a"]], [float(v) for v in g["b"]],
                            [float(v) for v in g["c"]])
    np.testing.assert_allclose(fac.bh, [float(v) for v in g["bhat"]], rtol=4e-16)
    np.testing.assert_allclose(fac.ch[:3], [float(v) for v in g["chat"]], rtol=4e-16)
    np.testing.assert_array_equal(fac.a, [-0.5] * 4)          # a is untouched (Alg. 1)
    x = oracle.tri_solve(fac, [float(v) for v in g["d"]])
    np.testing.assert_allclose(x, [float(v) for v in g["x"]], rtol=1e-15)


def test_exact_rational_random_small():
    """Asymmetric, row-varying diagonals: a transposed operand or an off-by-one index fails."""
    rng = np.random.default_rng(7)
    for n in (2, 3, 5, 7):
        a = rng.integers(-3, 4, n).astype(float)
        c = rng.integers(-3, 4, n).astype(float)
        b = (np.abs(a) + np.abs(c) + rng.integers(1, 4, n)).astype(float)
        d = rng.integers(-9, 10, n).astype(float)
        xe = exact_solve(dense_from_bands(n, tri_bands(a, b, c)), d)
        x = oracle.tri_solve(oracle.tri_factor(a, b, c), d)
        np.testing.assert_allclose(x, [float(v) for v in xe], rtol=0, atol=1e-14)


# --- closed forms ------------------------------------------------------------------------------

def test_factor_limit_closed_form():
    """b^_i -> (2+sqrt3)/2, c^_i -> -(2-sqrt3) for tridiag(-1/2, 2, -1/2) (fixed point of eq. 2)."""
    fac = oracle.tri_factor(*toeplitz_tri(64, 0.5))
    np.testing.assert_allclose(fac.bh[:4], [2.0, 1.875, 28 / 15, 209 / 112], rtol=4e-16)
    assert abs(fac.bh[40] - (2 + np.sqrt(3)) / 2) < 1e-15
    assert abs(fac.ch[40] + (2 - np.sqrt(3))) < 1e-15


@pytest.mark.parametrize("n", [5, 64, 512])
def test_toeplitz_eigenpairs(n):
    """tridiag(-r,1+2r,-r) v_k = lambda_k v_k, v_k(i)=sin(i k pi/(n+1)), lambda_k=1+4r sin^2(k pi/(2(n+1)))."""
    r = 0.5
    fac = oracle.tri_factor(*toeplitz_tri(n, r))
    i = np.arange(1, n + 1)
    for k in (1, 2, n // 2, n):
        v = np.sin(((i * k) % (2 * (n + 1))) * np.pi / (n + 1))     # exact integer range reduction
        lam = 1 + 4 * r * np.sin(k * np.pi / (2 * (n + 1))) ** 2
        x = oracle.tri_solve(fac, v)
        np.testing.assert_allclose(x, v / lam, rtol=0, atol=5e-15)


def test_config2_modal_decay_100_steps():
    """Config 2 (backward Euler diffusion): after 100 solves each sine mode has decayed by lambda_k^-100."""
    n, M, r, steps = 512, 6, 0.5, 100
    rng = np.random.default_rng(3)
    i = np.arange(1, n + 1)[:, None]
    ks = rng.integers(1, 17, size=(4, M))
    amps = rng.uniform(-1, 1, size=(4, M))
    u0 = sum(amps[m] * np.sin(ks[m] * np.pi * i / (n + 1)) for m in range(4))
    lam = 1 + 4 * r * np.sin(ks * np.pi / (2 * (n + 1))) ** 2
    expect = sum(amps[m] * lam[m] ** (-steps) * np.sin(ks[m] * np.pi * i / (n + 1)) for m in range(4))
    u = np.ascontiguousarray(u0)
    oracle.tri_solve_interleaved(oracle.tri_factor(*toeplitz_tri(n, r)), u, nsteps=steps)
    assert np.max(np.abs(u - expect)) < 1e-13
    # decay factors quoted in SURVEY 8(c): 0.99813 (k=1) .. 0.61971 (k=16)
    l1 = 1 + 2 * np.sin(np.pi / 1026) ** 2
    l16 = 1 + 2 * np.sin(16 * np.pi / 1026) ** 2
    assert abs(l1 ** -100 - 0.99813) < 1e-5 and abs(l16 ** -100 - 0.61971) < 1e-5


# --- library routine / invariants --------------------------------------------------------------

@pytest.mark.parametrize("n", [1, 2, 3, 4, 8, 33])
def test_against_dense_lapack(n):
    rng = np.random.default_rng(100 + n)
    a, c = rng.uniform(-1, 1, n), rng.uniform(-1, 1, n)
    b = np.abs(a) + np.abs(c) + rng.uniform(0.5, 1.5, n)
    b *= rng.choice([-1.0, 1.0], n)
    d = rng.uniform(-1, 1, n)
    A = np_dense_from_bands(n, tri_bands(a, b, c))
    x = oracle.tri_solve(oracle.tri_factor(a, b, c), d)
    np.testing.assert_allclose(x, np.linalg.solve(A, d), rtol=0, atol=1e-13)


def test_never_read_entries():
    """a_1 and c_N are outside the matrix: NaN there must not matter."""
    a, b, c = toeplitz_tri(6, 0.5)
    a[0] = np.nan
    c[-1] = np.nan
    d = np.arange(1.0, 7.0)
    x = oracle.tri_solve(oracle.tri_factor(a, b, c), d)
    a0, b0, c0 = toeplitz_tri(6, 0.5)
    np.testing.assert_array_equal(x, oracle.tri_solve(oracle.tri_factor(a0, b0, c0), d))
    assert np.all(np.isfinite(x))


@pytest.mark.parametrize("n", [64, 1024])
def test_residual_large(n):
    a, b, c = toeplitz_tri(n, 0.5)
    d = np.random.default_rng(n).uniform(-1, 1, n)
    x = oracle.tri_solve(oracle.tri_factor(a, b, c), d)
    res = b * x
    res[1:] += a[1:] * x[:-1]
    res[:-1] += c[:-1] * x[1:]
    assert np.max(np.abs(res - d)) < 1e-15 * 3 * 4      # few ulp * ||A|| * ||x||


def test_special_case_diagonal():
    n = 9
    b = np.linspace(1, 3, n)
    d = np.linspace(-2, 5, n)
    x = oracle.tri_solve(oracle.tri_factor(np.zeros(n), b, np.zeros(n)), d)
    np.testing.assert_array_equal(x, d / b)


def test_zero_pivot_reports_row():
    with pytest.raises(oracle.FactorError) as ei:
        oracle.tri_factor([0, 1, 1], [1, 1, 1], [1, 1, 0])     # b^_2 = 1 - 1*1 = 0
    assert ei.value.row == 2
    with pytest.raises(oracle.FactorError) as ei:
        oracle.tri_factor([0.0], [0.0], [0.0])
    assert ei.value.row == 1


# --- interleaved layout (Alg. 2 rowID +- M) -----------------------------------------

def test_interleaved_layout_and_subset():
    n, M = 7, 11
    rng = np.random.default_rng(5)
    a, c = rng.uniform(-1, 1, n), rng.uniform(-1, 1, n)
    b = 3 + rng.uniform(0, 1, n)
    fac = oracle.tri_factor(a, b, c)
    rhs = rng.uniform(-1, 1, (n, M))
    flat = rhs.copy().reshape(-1)                 # element i of system j at i*M + j
    expect = np.stack([oracle.tri_solve(fac, flat[j::M]) for j in range(M)], axis=1)
    out = rhs.copy()
    oracle.tri_solve_interleaved(fac, out)
    np.testing.assert_array_equal(out, expect)
    out1 = rhs.copy()
    oracle.tri_solve_interleaved(fac, out1, nthreads=1)
    np.testing.assert_array_equal(out1, expect)
    sub = rhs.copy()
    oracle.tri_solve_interleaved(fac, sub, subset=(1, 10, 3))       # systems 1, 4, 7
    touched = np.zeros(M, bool)
    touched[[1, 4, 7]] = True
    np.testing.assert_array_equal(sub[:, touched], expect[:, touched])
    np.testing.assert_array_equal(sub[:, ~touched], rhs[:, ~touched])
    two = rhs.copy()
    oracle.tri_solve_interleaved(fac, two, nsteps=2)
    once_more = expect.copy()
    oracle.tri_solve_interleaved(fac, once_more)
    np.testing.assert_array_equal(two, once_more)


def test_storage_formula():
    """one factor copy is 3N values against 4MN for per-system copies."""
    fac = oracle.tri_factor(*toeplitz_tri(64, 0.5))
    assert fac.a.size + fac.bh.size + fac.ch.size == 3 * 64
    M, N = 2 ** 16, 64
    assert abs(1 - (3 * N + M * N) / (4 * M * N) - 0.75) < 1e-4
