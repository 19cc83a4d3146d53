"""Pins for the oracle's periodic tridiagonal solve (Sec. 3.3, eq. 12-15:
Sherman-Morrison).  None of them retypes the oracle's formula: the splitting is checked entrywise
against the cyclic matrix, the solve against dense LAPACK solves and an exact rational solve, against
the closed-form eigenpairs of circulant matrices, and against conservation of the column sum."""
from fractions import Fraction

import numpy as np
import pytest

import oracle
from tests._exact import exact_solve


def cyclic_dense(a, b, c):
    n = len(b)
    A = np.zeros((n, n))
    for i in range(n):
        A[i, i] += b[i]
        A[i, (i - 1) % n] += a[i]
        A[i, (i + 1) % n] += c[i]
    return A


def test_splitting_equals_cyclic_matrix():
    """eq. 12-13: A' + u (x) v must equal the periodic matrix entry by entry (rebuilt from the paper's
    definitions of A', u, v with constant diagonals, independent of the oracle)."""
    n, a, b, c = 7, -0.3, 2.1, -0.7
    A = cyclic_dense([a] * n, [b] * n, [c] * n)
    Ap = np.diag([b] * n) + np.diag([a] * (n - 1), -1) + np.diag([c] * (n - 1), 1)
    Ap[0, 0] = 2 * b
    Ap[-1, -1] = b + a * c / b
    u = np.zeros(n); u[0] = -b; u[-1] = c
    v = np.zeros(n); v[0] = 1.0; v[-1] = -a / b
    assert np.allclose(Ap + np.outer(u, v), A, rtol=0, atol=1e-15)
    # the oracle's factor data describe the same splitting: z = A'^{-1} u, den = 1 + v.z
    f = oracle.tri_periodic_factor([a] * n, [b] * n, [c] * n)
    assert np.allclose(Ap @ f.z, u, atol=1e-14)
    assert abs(f.vN - v[-1]) < 1e-16 and abs(f.den - (1 + v @ f.z)) < 1e-14


@pytest.mark.parametrize("n", [3, 4, 5, 8, 33])
def test_dense_solve_random_cyclic(n):
    rng = np.random.default_rng(n)
    a, c = rng.uniform(-1, 1, n), rng.uniform(-1, 1, n)
    b = np.abs(a) + np.abs(c) + rng.uniform(0.5, 1.5, n)
    d = rng.uniform(-1, 1, n)
    x = oracle.tri_periodic_solve(oracle.tri_periodic_factor(a, b, c), d)
    ref = np.linalg.solve(cyclic_dense(a, b, c), d)
    assert np.max(np.abs(x - ref)) <= 1e-13 * max(1.0, np.max(np.abs(ref)))
    # residual against the cyclic matrix itself
    assert np.max(np.abs(cyclic_dense(a, b, c) @ x - d)) <= 1e-13


def test_exact_rational_example():
    """N = 5, a = c = -1/2, b = 2 (I + r*periodic Laplacian, r = 1/2), d = (1,2,3,4,5): exact Gaussian
    elimination in rationals on the cyclic matrix."""
    n = 5
    A = [[Fraction(0)] * n for _ in range(n)]
    for i in range(n):
        A[i][i] = Fraction(2)
        A[i][(i - 1) % n] += Fraction(-1, 2)
        A[i][(i + 1) % n] += Fraction(-1, 2)
    exact = exact_solve(A, [Fraction(k) for k in range(1, 6)])
    x = oracle.tri_periodic_solve(oracle.tri_periodic_factor([-0.5] * n, [2.0] * n, [-0.5] * n),
                                  np.arange(1.0, 6.0))
    assert np.max(np.abs(x - np.array([float(e) for e in exact]))) <= 4e-16 * 5
    assert sum(exact) == Fraction(15)  # column sums of A are 1: the sum is conserved exactly


@pytest.mark.parametrize("n", [8, 64, 512])
def test_circulant_eigenpairs(n):
    """Circulant tridiag(-r, 1+2r, -r): eigenvectors cos/sin(2 pi k j / n), eigenvalues
    1 + 4 r sin^2(pi k / n) (textbook); solving with an eigenvector must scale it by 1/lambda."""
    r = 0.5
    f = oracle.tri_periodic_factor([-r] * n, [1 + 2 * r] * n, [-r] * n)
    j = np.arange(n)
    for k in (0, 1, 3, n // 2):
        lam = 1 + 4 * r * np.sin(np.pi * k / n) ** 2
        for mode in (np.cos(2 * np.pi * k * j / n), np.sin(2 * np.pi * k * j / n)):
            x = oracle.tri_periodic_solve(f, mode)
            assert np.max(np.abs(x - mode / lam)) <= 1e-13


def test_mass_conserved_over_steps_interleaved():
    """Implicit periodic diffusion conserves the mean (PAPER.md:339-348 holds for periodic BCs): the
    column sums of I + r*L_per are 1, so sum(x) == sum(d) every step; and the interleaved driver equals
    the per-system routine."""
    n, M, r, steps = 64, 37, 0.5, 25
    rng = np.random.default_rng(1)
    rhs = rng.uniform(-1, 1, (n, M))
    f = oracle.tri_periodic_factor([-r] * n, [1 + 2 * r] * n, [-r] * n)
    out = rhs.copy()
    oracle.tri_periodic_solve_interleaved(f, out, nsteps=steps)
    assert np.max(np.abs(out.sum(axis=0) - rhs.sum(axis=0))) <= 1e-12
    col = rhs[:, 5].copy()
    for _ in range(steps):
        col = oracle.tri_periodic_solve(f, col)
    assert np.array_equal(col, out[:, 5])
    # exact modal decay of the k = 2 cosine over `steps` steps
    mode = np.cos(2 * np.pi * 2 * np.arange(n) / n)[:, None].copy()
    oracle.tri_periodic_solve_interleaved(f, mode, nsteps=steps)
    lam = 1 + 4 * r * np.sin(np.pi * 2 / n) ** 2
    assert np.max(np.abs(mode[:, 0] - np.cos(2 * np.pi * 2 * np.arange(n) / n) * lam ** -steps)) <= 1e-13


def test_bad_inputs():
    with pytest.raises(oracle.FactorError):
        oracle.tri_periodic_factor([1.0, 1.0], [2.0, 2.0], [1.0, 1.0])  # n < 3
    with pytest.raises(oracle.FactorError):
        oracle.tri_periodic_factor([1.0] * 4, [0.0, 2.0, 2.0, 2.0], [1.0] * 4)  # b_1 = 0


# ---- Crank-Nicolson diffusion step (eq. 9-11) -----------------------------------------

def test_cn_periodic_modal_amplification_and_mass():
    """Periodic CN: the mode cos(2 pi k j / N) is multiplied per step by
    (1 - 4 s sin^2(pi k / N)) / (1 + 4 s sin^2(pi k / N)), s = sigma_x (von Neumann factor of eq. 9); the
    sum over the grid is conserved (column sums of both stencils are 1)."""
    n, M, s, steps = 64, 5, 0.7, 30
    j = np.arange(n)
    u = np.zeros((n, M))
    ks = [0, 1, 3, 7, 31]
    for m, k in enumerate(ks):
        u[:, m] = np.cos(2 * np.pi * k * j / n)
    u0 = u.copy()
    f = oracle.tri_periodic_factor([-s] * n, [1 + 2 * s] * n, [-s] * n)
    oracle.tri_cn_step_interleaved(f, u, s, 1 - 2 * s, s, nsteps=steps)
    for m, k in enumerate(ks):
        q = 4 * s * np.sin(np.pi * k / n) ** 2
        assert np.max(np.abs(u[:, m] - u0[:, m] * ((1 - q) / (1 + q)) ** steps)) <= 1e-13
    rng = np.random.default_rng(4)
    w = rng.uniform(-1, 1, (n, 3))
    w0 = w.copy()
    oracle.tri_cn_step_interleaved(f, w, s, 1 - 2 * s, s, nsteps=steps)
    assert np.max(np.abs(w.sum(axis=0) - w0.sum(axis=0))) <= 1e-13


@pytest.mark.parametrize("periodic", [False, True])
def test_cn_step_dense_restatement(periodic):
    """One step against numpy: (I - s L) u' = (I + s L) u with L the (periodic | truncated) second difference."""
    n, s = 12, 0.4
    I = np.eye(n)
    L = -2 * I + np.diag(np.ones(n - 1), 1) + np.diag(np.ones(n - 1), -1)
    if periodic:
        L[0, -1] = L[-1, 0] = 1.0
    rng = np.random.default_rng(5)
    u = rng.uniform(-1, 1, (n, 4))
    ref = np.linalg.solve(I - s * L, (I + s * L) @ u)
    f = (oracle.tri_periodic_factor if periodic else oracle.tri_factor)([-s] * n, [1 + 2 * s] * n, [-s] * n)
    assert np.max(np.abs(oracle.tri_explicit(u[:, 0], s, 1 - 2 * s, s, periodic) - ((I + s * L) @ u)[:, 0])) <= 1e-15
    oracle.tri_cn_step_interleaved(f, u, s, 1 - 2 * s, s)
    assert np.max(np.abs(u - ref)) <= 1e-14
