"""Pins for the oracle's cyclic pentadiagonal solve (eq. 26a; the paper cites [24,4,25]
for the method, the oracle reaches x = A^{-1} f by a Woodbury correction -- DESIGN.md C-31) and for the
periodic Cahn-Hilliard step.  Independent checks: dense and exact-rational solves of
the cyclic matrix, circulant eigenpairs, exact conservation of mass under periodic BCs (eq. 21-22)."""
from fractions import Fraction

import numpy as np
import pytest

import oracle
from tests._exact import exact_solve


def cyclic_dense(a, b, c, d, e):
    n = len(c)
    A = np.zeros((n, n))
    for i in range(n):
        for off, v in ((-2, a), (-1, b), (0, c), (1, d), (2, e)):
            A[i, (i + off) % n] += v[i]
    return A


@pytest.mark.parametrize("n", [5, 6, 7, 8, 33, 64])
def test_dense_solve_random_cyclic(n):
    rng = np.random.default_rng(n)
    a, b, d, e = (rng.uniform(-1, 1, n) for _ in range(4))
    c = np.abs(a) + np.abs(b) + np.abs(d) + np.abs(e) + rng.uniform(0.5, 1.5, n)
    f = rng.uniform(-1, 1, n)
    x = oracle.penta_periodic_solve(oracle.penta_periodic_factor(a, b, c, d, e), f)
    A = cyclic_dense(a, b, c, d, e)
    ref = np.linalg.solve(A, f)
    assert np.max(np.abs(x - ref)) <= 1e-13 * max(1.0, np.max(np.abs(ref)))
    assert np.max(np.abs(A @ x - f)) <= 1e-13


def test_exact_rational_example():
    """N = 6, I + (1/2)*periodic [1,-4,6,-4,1], f = (1..6): exact rational elimination on the cyclic matrix."""
    n = 6
    st = {-2: Fraction(1, 2), -1: Fraction(-2), 0: Fraction(4), 1: Fraction(-2), 2: Fraction(1, 2)}
    A = [[Fraction(0)] * n for _ in range(n)]
    for i in range(n):
        for off, v in st.items():
            A[i][(i + off) % n] += v
    exact = exact_solve(A, [Fraction(k) for k in range(1, n + 1)])
    x = oracle.penta_periodic_solve(
        oracle.penta_periodic_factor([0.5] * n, [-2.0] * n, [4.0] * n, [-2.0] * n, [0.5] * n), np.arange(1.0, n + 1))
    assert np.max(np.abs(x - np.array([float(v) for v in exact]))) <= 1e-14
    assert sum(exact) == Fraction(21)  # column sums are 1


@pytest.mark.parametrize("n", [8, 64, 256])
def test_circulant_eigenpairs(n):
    """Circulant I + r*[1,-4,6,-4,1]: eigenvalues 1 + 16 r sin^4(pi k / n) on cos/sin(2 pi k j / n)."""
    r = 0.5
    f = oracle.penta_periodic_factor([r] * n, [-4 * r] * n, [1 + 6 * r] * n, [-4 * r] * n, [r] * n)
    j = np.arange(n)
    for k in (0, 1, 2, n // 2):
        lam = 1 + 16 * r * np.sin(np.pi * k / n) ** 4
        for mode in (np.cos(2 * np.pi * k * j / n), np.sin(2 * np.pi * k * j / n)):
            assert np.max(np.abs(oracle.penta_periodic_solve(f, mode) - mode / lam)) <= 1e-13


def test_ch_rhs_periodic_is_circulant_stencil():
    n, alpha = 16, 0.3
    rng = np.random.default_rng(2)
    c = rng.uniform(-1, 1, n)
    w = c ** 3 - c
    D2 = -2 * np.eye(n) + np.roll(np.eye(n), 1, axis=1) + np.roll(np.eye(n), -1, axis=1)
    assert np.max(np.abs(oracle.ch_rhs_periodic(c, alpha) - (c + alpha * (D2 @ w)))) <= 1e-15


def test_periodic_ch_conserves_mass_and_matches_dense_model():
    """PAPER.md:339-348 (eq. 21-22): with periodic BCs d<C>/dt = 0.  Discretely: column sums of the
    circulant D2 are 0 and of I + sigma*D4 are 1, so sum(c) is conserved to rounding every step.  The
    stepper is also compared with a dense restatement of eq. 24 (numpy solve of the circulant system)."""
    n, M, steps = 32, 9, 50
    sigma, alpha = 1.3778768139120494, 0.08300231363980311
    rng = np.random.default_rng(3)
    c0 = 0.1 * rng.uniform(-1, 1, (n, M))
    f = oracle.penta_periodic_factor([sigma] * n, [-4 * sigma] * n, [1 + 6 * sigma] * n, [-4 * sigma] * n, [sigma] * n)
    c = c0.copy()
    oracle.ch_periodic_step_interleaved(f, c, alpha, nsteps=steps)
    assert np.max(np.abs(c.sum(axis=0) - c0.sum(axis=0))) <= 1e-14
    I = np.eye(n)
    D2 = -2 * I + np.roll(I, 1, axis=1) + np.roll(I, -1, axis=1)
    A = I + sigma * (D2 @ D2)
    ref = c0.copy()
    for _ in range(steps):
        ref = np.linalg.solve(A, ref + alpha * (D2 @ (ref ** 3 - ref)))
    assert np.max(np.abs(c - ref)) <= 1e-13
    # nsteps solves in mode 0 equal repeated single solves
    x = c0[:, 0].copy()
    for _ in range(3):
        x = oracle.penta_periodic_solve(f, x)
    y = c0.copy()
    oracle.penta_periodic_solve_interleaved(f, y, nsteps=3)
    assert np.array_equal(x, y[:, 0])


def test_bad_inputs():
    with pytest.raises(oracle.FactorError):
        oracle.penta_periodic_factor(*([[1.0] * 4] * 5))  # n < 5


# ---- Crank-Nicolson hyperdiffusion step (eq. 17-19) -----------------------------------

def test_cn_hyperdiffusion_modal_amplification_and_mass():
    """Periodic CN hyperdiffusion: cos(2 pi k j / N) is multiplied per step by (1 - q)/(1 + q),
    q = 16 s sin^4(pi k / N) (symbol of the five-point stencil of eq. 18); the grid sum is conserved."""
    n, s, steps = 64, 0.3, 20
    j = np.arange(n)
    ks = [0, 1, 2, 5, 31]
    u = np.stack([np.cos(2 * np.pi * k * j / n) for k in ks], axis=1).copy()
    u0 = u.copy()
    f = oracle.penta_periodic_factor([s] * n, [-4 * s] * n, [1 + 6 * s] * n, [-4 * s] * n, [s] * n)
    x5 = [-s, 4 * s, 1 - 6 * s, 4 * s, -s]
    oracle.penta_cn_step_interleaved(f, u, x5, nsteps=steps)
    for m, k in enumerate(ks):
        q = 16 * s * np.sin(np.pi * k / n) ** 4
        assert np.max(np.abs(u[:, m] - u0[:, m] * ((1 - q) / (1 + q)) ** steps)) <= 1e-13
    rng = np.random.default_rng(6)
    w = rng.uniform(-1, 1, (n, 3))
    w0 = w.copy()
    oracle.penta_cn_step_interleaved(f, w, x5, nsteps=steps)
    assert np.max(np.abs(w.sum(axis=0) - w0.sum(axis=0))) <= 1e-13


@pytest.mark.parametrize("periodic", [False, True])
def test_cn_hyperdiffusion_dense_restatement(periodic):
    n, s = 12, 0.4
    I = np.eye(n)
    L = -2 * I + np.diag(np.ones(n - 1), 1) + np.diag(np.ones(n - 1), -1)
    if periodic:
        L[0, -1] = L[-1, 0] = 1.0
        D4 = L @ L
    else:
        D4 = np.zeros((n, n))   # truncated [1,-4,6,-4,1] (ghost values zero), not L @ L (C-25)
        for i in range(n):
            for o, v in ((-2, 1.0), (-1, -4.0), (0, 6.0), (1, -4.0), (2, 1.0)):
                if 0 <= i + o < n:
                    D4[i, i + o] = v
    rng = np.random.default_rng(7)
    u = rng.uniform(-1, 1, (n, 4))
    ref = np.linalg.solve(I + s * D4, (I - s * D4) @ u)
    st = ([s] * n, [-4 * s] * n, [1 + 6 * s] * n, [-4 * s] * n, [s] * n)
    f = (oracle.penta_periodic_factor if periodic else oracle.penta_factor)(*st)
    x5 = [-s, 4 * s, 1 - 6 * s, 4 * s, -s]
    assert np.max(np.abs(oracle.penta_explicit(u[:, 0], x5, periodic) - ((I - s * D4) @ u)[:, 0])) <= 1e-15
    oracle.penta_cn_step_interleaved(f, u, x5)
    assert np.max(np.abs(u - ref)) <= 1e-13
