"""Pins for the pentadiagonal oracle (orc_penta_factor / orc_penta_solve), paper naming a..e.

Expected values come from exact rational elimination, numpy dense solves, L*R rebuilt densely,
closed-form eigenpairs of I + r*T^2 and reductions to the tridiagonal routine.  No GPU needed.
"""
import os

import numpy as np
import pytest

import oracle
from tests._exact import dense_from_bands, exact_solve, np_dense_from_bands, read_golden


def penta_bands(a, b, c, d, e):
    return {-2: a, -1: b, 0: c, 1: d, 2: e}


def toeplitz_penta(n, r):
    """I + r*[1,-4,6,-4,1], truncated at both ends (BASELINE config 3)."""
    return (np.full(n, r), np.full(n, -4 * r), np.full(n, 1 + 6 * r), np.full(n, -4 * r),
            np.full(n, r))


def random_penta(n, rng, dominant=True):
    a, b, d, e = (rng.uniform(-1, 1, n) for _ in range(4))
    c = rng.uniform(0.5, 1.5, n) * rng.choice([-1.0, 1.0], n)
    if dominant:
        c = c + np.sign(c) * (np.abs(a) + np.abs(b) + np.abs(d) + np.abs(e))
    return a, b, c, d, e


# --- worked example ----------------------------------------------------------------------------

def test_worked_example_n5(golden_dir):
    g = read_golden(os.path.join(golden_dir, "penta_n5.txt"))
    n = 5
    A = dense_from_bands(n, penta_bands(g["a"], g["b"], g["c"], g["d"], g["e"]))
    assert exact_solve(A, g["f"]) == g["x"]
    # the fixture's factor values satisfy L*R == A exactly (eq. 16a-b)
    eps, beta = [None, None] + g["a"][2:], [None] + g["beta"]
    for i in range(n):
        for j in range(n):
            s = 0
            for k in range(n):                 # L[i][k] * R[k][j]
                L = g["alpha"][i] if k == i else beta[i] if k == i - 1 else eps[i] if k == i - 2 else 0
                R = 1 if j == k else g["gamma"][k] if (j == k + 1 and k < n - 1) else \
                    g["delta"][k] if (j == k + 2 and k < n - 2) else 0
                s += L * R
            assert s == A[i][j]
    fl = lambda key: [float(v) for v in g[key]]
    fac = oracle.penta_factor(fl("a"), fl("b"), fl("c"), fl("d"), fl("e"))
    np.testing.assert_allclose(fac.alpha, fl("alpha"), rtol=1e-15)
    np.testing.assert_allclose(fac.beta[1:], fl("beta"), rtol=1e-15)
    np.testing.assert_allclose(fac.gamma[:4], fl("gamma"), rtol=1e-15)
    np.testing.assert_allclose(fac.delta[:3], fl("delta"), rtol=1e-15)
    np.testing.assert_array_equal(fac.eps, fl("a"))           # step 14: eps_i = a_i
    np.testing.assert_allclose(oracle.penta_solve(fac, fl("f")), fl("x"), rtol=2e-15)


def test_exact_rational_random_small():
    rng = np.random.default_rng(11)
    for n in (1, 2, 3, 4, 5, 6, 8):
        a, b, d, e = (rng.integers(-3, 4, n).astype(float) for _ in range(4))
        c = (np.abs(a) + np.abs(b) + np.abs(d) + np.abs(e) + rng.integers(1, 4, n)).astype(float)
        f = rng.integers(-9, 10, n).astype(float)
        xe = exact_solve(dense_from_bands(n, penta_bands(a, b, c, d, e)), f)
        x = oracle.penta_solve(oracle.penta_factor(a, b, c, d, e), f)
        np.testing.assert_allclose(x, [float(v) for v in xe], rtol=0, atol=2e-14)


# --- structure -----------------------------------------------------------------------------------

@pytest.mark.parametrize("n", [4, 5, 7, 8, 40])
def test_LR_rebuild(n):
    """Rebuild L (eps, beta, alpha) and unit-upper R (gamma, delta) densely: L @ R == A."""
    rng = np.random.default_rng(n)
    a, b, c, d, e = random_penta(n, rng)
    fac = oracle.penta_factor(a, b, c, d, e)
    L = np_dense_from_bands(n, {-2: fac.eps, -1: fac.beta, 0: fac.alpha})
    R = np_dense_from_bands(n, {0: np.ones(n), 1: fac.gamma, 2: fac.delta})
    np.testing.assert_allclose(L @ R, np_dense_from_bands(n, penta_bands(a, b, c, d, e)),
                               rtol=0, atol=1e-14)


@pytest.mark.parametrize("n", [4, 5, 6, 9, 64])
def test_general_form_is_bitwise_the_literal_steps(n):
    """[C-13]: the guarded general-row recurrences reproduce Sec. 4.1 steps 1-14 exactly for N >= 4."""
    rng = np.random.default_rng(50 + n)
    diags = random_penta(n, rng)
    lit = oracle.penta_factor(*diags)
    gen = oracle.penta_factor(*diags, general=True)
    for k in ("eps", "beta", "alpha", "gamma", "delta"):
        np.testing.assert_array_equal(getattr(lit, k), getattr(gen, k))


def test_never_read_entries():
    n = 7
    a, b, c, d, e = toeplitz_penta(n, 0.5)
    ref = oracle.penta_solve(oracle.penta_factor(a, b, c, d, e), np.arange(1.0, n + 1))
    a[0] = a[1] = b[0] = d[-1] = e[-1] = e[-2] = np.nan
    x = oracle.penta_solve(oracle.penta_factor(a, b, c, d, e), np.arange(1.0, n + 1))
    np.testing.assert_array_equal(x, ref)


# --- library routine ---------------------------------------------------------------------------------

@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 8, 33])
@pytest.mark.parametrize("dominant", [True, False])
def test_against_dense_lapack(n, dominant):
    rng = np.random.default_rng(1000 + n)
    if dominant:
        a, b, c, d, e = random_penta(n, rng)
    else:                                   # SPD but not diagonally dominant (config 3 / 5 like)
        a, b, c, d, e = toeplitz_penta(n, 1.3778768139120494)
    f = rng.uniform(-1, 1, n)
    x = oracle.penta_solve(oracle.penta_factor(a, b, c, d, e), f)
    A = np_dense_from_bands(n, penta_bands(a, b, c, d, e))
    np.testing.assert_allclose(x, np.linalg.solve(A, f), rtol=0, atol=2e-13)


# --- closed forms --------------------------------------------------------------------------------

def test_factor_limit_closed_form():
    """Fixed point for I + 1/2*[1,-4,6,-4,1]: alpha -> 3/2+sqrt2, beta -> -(1+sqrt2/2),
    gamma -> -(2-sqrt2), delta -> 3-2sqrt2."""
    fac = oracle.penta_factor(*toeplitz_penta(96, 0.5))
    s2 = np.sqrt(2.0)
    assert abs(fac.alpha[60] - (1.5 + s2)) < 2e-15
    assert abs(fac.beta[60] + (1 + s2 / 2)) < 2e-15
    assert abs(fac.gamma[60] + (2 - s2)) < 2e-15
    assert abs(fac.delta[60] - (3 - 2 * s2)) < 2e-15


def i_plus_r_T2(n, r):
    """I + r*T^2, T = tridiag(-1,2,-1): the Toeplitz penta bands with corner entries 1+5r [C-25]."""
    a, b, c, d, e = toeplitz_penta(n, r)
    c[0] = c[-1] = 1 + 5 * r
    return a, b, c, d, e


def test_T2_identity():
    n, r = 9, 0.5
    T = np_dense_from_bands(n, {-1: -np.ones(n), 0: 2 * np.ones(n), 1: -np.ones(n)})
    np.testing.assert_allclose(np.eye(n) + r * T @ T,
                               np_dense_from_bands(n, penta_bands(*i_plus_r_T2(n, r))), atol=1e-15)


@pytest.mark.parametrize("n", [6, 64, 512])
def test_toeplitz_eigenpairs(n):
    """(I + r T^2) v_k = lambda_k v_k, v_k(i) = sin(i k pi/(n+1)), lambda_k = 1 + 16 r sin^4(k pi/(2(n+1)))."""
    r = 0.5
    fac = oracle.penta_factor(*i_plus_r_T2(n, r))
    i = np.arange(1, n + 1)
    for k in (1, 3, n // 2, n):
        v = np.sin(((i * k) % (2 * (n + 1))) * np.pi / (n + 1))
        lam = 1 + 16 * r * np.sin(k * np.pi / (2 * (n + 1))) ** 4
        np.testing.assert_allclose(oracle.penta_solve(fac, v), v / lam, rtol=0, atol=1e-14)


def test_modal_decay_100_steps():
    n, r, steps, M = 512, 0.5, 100, 5
    fac = oracle.penta_factor(*i_plus_r_T2(n, r))
    i = np.arange(1, n + 1)[:, None]
    ks = np.array([1, 7, 16, 100, 300])[None, :]
    u = np.ascontiguousarray(np.sin(((i * ks) % (2 * (n + 1))) * np.pi / (n + 1)))
    expect = u * (1 + 16 * r * np.sin(ks * np.pi / (2 * (n + 1))) ** 4) ** (-steps)
    oracle.penta_solve_interleaved(fac, u, nsteps=steps)
    assert np.max(np.abs(u - expect)) < 1e-13
    assert u.shape == (n, M)


def test_config3_norm_non_increasing():
    """Config-3 LHS is SPD with spectrum in [1, 9]: ||u^{n+1}||_2 <= ||u^n||_2 for every system."""
    n, M = 512, 4
    fac = oracle.penta_factor(*toeplitz_penta(n, 0.5))
    A = np_dense_from_bands(n, penta_bands(*toeplitz_penta(n, 0.5)))
    ev = np.linalg.eigvalsh(A)
    assert ev[0] >= 1 - 1e-12 and ev[-1] <= 9 + 1e-12
    u = np.random.default_rng(0).uniform(-1, 1, (n, M))
    prev = np.linalg.norm(u, axis=0)
    for _ in range(100):
        oracle.penta_solve_interleaved(fac, u)
        cur = np.linalg.norm(u, axis=0)
        assert np.all(cur <= prev)
        prev = cur


# --- reductions --------------------------------------------------------------------------------------

def test_reduces_to_tridiagonal():
    n = 17
    rng = np.random.default_rng(4)
    b, d = rng.uniform(-1, 1, n), rng.uniform(-1, 1, n)
    c = 3 + rng.uniform(0, 1, n)
    f = rng.uniform(-1, 1, n)
    z = np.zeros(n)
    xp = oracle.penta_solve(oracle.penta_factor(z, b, c, d, z), f)
    xt = oracle.tri_solve(oracle.tri_factor(b, c, d), f)
    np.testing.assert_allclose(xp, xt, rtol=0, atol=1e-15)


def test_zero_pivot_reports_row():
    with pytest.raises(oracle.FactorError) as ei:
        oracle.penta_factor([0] * 5, [0, 1, 0, 0, 0], [1, 1, 1, 1, 1], [1, 0, 0, 0, 0], [0] * 5)
    assert ei.value.row == 2                                 # alpha_2 = 1 - 1*1


def test_interleaved_layout():
    n, M = 6, 9
    rng = np.random.default_rng(8)
    fac = oracle.penta_factor(*random_penta(n, rng))
    rhs = rng.uniform(-1, 1, (n, M))
    expect = np.stack([oracle.penta_solve(fac, rhs[:, j]) for j in range(M)], axis=1)
    out = rhs.copy()
    oracle.penta_solve_interleaved(fac, out)
    np.testing.assert_array_equal(out, expect)


def test_storage_formula():
    """5N + MN against 6MN, about 83% less."""
    M, N = 2 ** 16, 256
    assert abs(1 - (5 * N + M * N) / (6 * M * N) - 5 / 6) < 1e-4
