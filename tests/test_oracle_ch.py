"""Pins for the Cahn-Hilliard explicit half and stepper (orc_ch_rhs, orc_ch_step_interleaved).

PAPER.md:365-392 (eq. 24-26c) with BASELINE config 5's truncated stencils [C-18].  Expected values
come from a dense restatement of eq. 24 (matrices D2, D4 written out from eq. 25a-b, numpy solve),
the exact discrete mass balance of that scheme [C-19] and special cases.  No GPU needed.
"""
import numpy as np
import pytest

import oracle
from tests._exact import np_dense_from_bands

G, L, N5, DT = 0.01, 2 * np.pi, 256, 5e-5


def ch_params(n=N5, length=L, dt=DT, g=G):
    dx = length / n
    return g * dt / dx ** 4, dt / dx ** 2          # sigma (eq. 26b), alpha (eq. 26c)


def ch_lhs(n, sigma):
    return (np.full(n, sigma), np.full(n, -4 * sigma), np.full(n, 1 + 6 * sigma),
            np.full(n, -4 * sigma), np.full(n, sigma))


def dense_D2(n):
    return np_dense_from_bands(n, {-1: np.ones(n), 0: -2 * np.ones(n), 1: np.ones(n)})


def dense_D4(n):
    return np_dense_from_bands(n, {-2: np.ones(n), -1: -4 * np.ones(n), 0: 6 * np.ones(n),
                                   1: -4 * np.ones(n), 2: np.ones(n)})


def test_config5_constants():
    """sigma, alpha quoted in SURVEY 8(a5) for g=0.01, L=2pi, N=256, dt=5e-5."""
    sigma, alpha = ch_params()
    assert abs(sigma - 1.3778768139120494) < 1e-14
    assert abs(alpha - 0.08300231363980311) < 1e-15


@pytest.mark.parametrize("n", [1, 2, 3, 8, 31])
def test_rhs_against_dense_stencil(n):
    rng = np.random.default_rng(n)
    c = rng.uniform(-1, 1, n)
    alpha = 0.37
    expect = c + alpha * dense_D2(n) @ (c ** 3 - c)
    np.testing.assert_allclose(oracle.ch_rhs(c, alpha), expect, rtol=0, atol=1e-15)


def test_rhs_hand_values():
    """n=3, c=(1,2,-1), alpha=1/2: w=(0,6,0); f = c + (w_{i-1}-2w_i+w_{i+1})/2 = (4,-4,2)."""
    np.testing.assert_array_equal(oracle.ch_rhs([1.0, 2.0, -1.0], 0.5), [4.0, -4.0, 2.0])


@pytest.mark.parametrize("n", [5, 16, 64])
def test_step_against_dense_restatement(n):
    """c^{n+1} = (I + sigma D4)^{-1} (c + alpha D2 (c^3 - c))  -- eq. 24 written with dense matrices."""
    sigma, alpha = ch_params(n=n, length=L * n / N5)          # same dx as config 5
    rng = np.random.default_rng(n)
    M, steps = 3, 4
    c = 0.1 * rng.uniform(-1, 1, (n, M))
    A = np.eye(n) + sigma * dense_D4(n)
    expect = c.copy()
    for _ in range(steps):
        expect = np.linalg.solve(A, expect + alpha * dense_D2(n) @ (expect ** 3 - expect))
    fac = oracle.penta_factor(*ch_lhs(n, sigma))
    got = c.copy()
    oracle.ch_step_interleaved(fac, got, alpha, nsteps=steps)
    np.testing.assert_allclose(got, expect, rtol=0, atol=1e-15)


def test_mass_balance_identity_truncated():
    """[C-19] column sums of truncated D2 / D4 give, every step,
    sum c^{n+1} - sum c^n = -alpha (w_1 + w_N)^n - sigma (3c_1 - c_2 - c_{N-1} + 3c_N)^{n+1}."""
    n, M = N5, 3
    sigma, alpha = ch_params()
    fac = oracle.penta_factor(*ch_lhs(n, sigma))
    c = 0.1 * np.random.default_rng(1).uniform(-1, 1, (n, M))
    for _ in range(25):
        w = c ** 3 - c
        new = c.copy()
        oracle.ch_step_interleaved(fac, new, alpha)
        lhs = new.sum(0) - c.sum(0)
        rhs = -alpha * (w[0] + w[-1]) - sigma * (3 * new[0] - new[1] - new[-2] + 3 * new[-1])
        assert np.max(np.abs(lhs - rhs)) < 5e-14
        c = new


def test_zero_state_and_linearisation():
    n = 32
    sigma, alpha = ch_params(n=n, length=L * n / N5)
    fac = oracle.penta_factor(*ch_lhs(n, sigma))
    z = np.zeros((n, 2))
    oracle.ch_step_interleaved(fac, z, alpha, nsteps=3)
    assert not z.any()
    # |c| << 1: the step is (I + sigma D4)^{-1} (I - alpha D2) c up to O(c^3)
    c = 1e-6 * np.random.default_rng(2).uniform(-1, 1, (n, 1))
    lin = np.linalg.solve(np.eye(n) + sigma * dense_D4(n), c - alpha * dense_D2(n) @ c)
    got = c.copy()
    oracle.ch_step_interleaved(fac, got, alpha)
    assert np.max(np.abs(got - lin)) < 1e-17


def test_config5_is_benign():
    """over 1000 steps (t = 0.05) max|c| stays of order 0.1 (no blow-up) and a 1e-15
    relative perturbation of c0 stays at rounding level (no chaos): the 1e-10 parity tolerance is safe."""
    sigma, alpha = ch_params()
    fac = oracle.penta_factor(*ch_lhs(N5, sigma))
    c = 0.1 * np.random.default_rng(0).uniform(-1, 1, (N5, 4))
    p = c * (1 + 1e-15)
    oracle.ch_step_interleaved(fac, c, alpha, nsteps=1000)
    oracle.ch_step_interleaved(fac, p, alpha, nsteps=1000)
    assert 0.03 < np.max(np.abs(c)) < 0.2
    assert np.max(np.abs(c - p)) / np.max(np.abs(c)) < 1e-13


def test_subset_and_threads():
    n, M = 16, 10
    sigma, alpha = ch_params(n=n, length=L * n / N5)
    fac = oracle.penta_factor(*ch_lhs(n, sigma))
    c = 0.1 * np.random.default_rng(9).uniform(-1, 1, (n, M))
    full = c.copy()
    oracle.ch_step_interleaved(fac, full, alpha, nsteps=2, nthreads=1)
    sub = c.copy()
    used = oracle.ch_step_interleaved(fac, sub, alpha, nsteps=2, subset=(2, 9, 2), nthreads=2)
    assert used == 2
    cols = [2, 4, 6, 8]
    np.testing.assert_array_equal(sub[:, cols], full[:, cols])
    rest = [j for j in range(M) if j not in cols]
    np.testing.assert_array_equal(sub[:, rest], c[:, rest])


# ---- coarsening statistic (eq. 30) ---------------------------------------------------

def test_lbar_closed_forms():
    """<C^2> of a constant c0 is c0^2; of A*cos(2 pi k x / L) on the periodic grid it is A^2 / 2 exactly
    (0 < k < N/2); the batch value is the mean of 1/(1 - <C^2>) over the runs."""
    import oracle
    n = 64
    j = np.arange(n)
    cols = [np.full(n, 0.3), 0.8 * np.cos(2 * np.pi * 5 * j / n), 0.5 * np.sin(2 * np.pi * 3 * j / n), np.zeros(n)]
    c = np.ascontiguousarray(np.stack(cols, axis=1))
    expect = np.mean([1 / (1 - 0.09), 1 / (1 - 0.32), 1 / (1 - 0.125), 1.0])
    assert abs(oracle.lbar_interleaved(c) - expect) <= 1e-15
    # a single run; and invariance under a permutation of the rows (it is a mean over the grid)
    one = np.ascontiguousarray(c[:, 1:2])
    assert abs(oracle.lbar_interleaved(one) - 1 / (1 - 0.32)) <= 1e-15
    assert abs(oracle.lbar_interleaved(np.ascontiguousarray(one[::-1])) - 1 / (1 - 0.32)) <= 1e-15
