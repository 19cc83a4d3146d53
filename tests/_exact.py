"""Exact rational arithmetic helpers for the oracle pins (independent of oracle/ and of the CUDA path)."""
from fractions import Fraction

import numpy as np


def dense_from_bands(n, bands):
    """bands: {offset: sequence of length n}; entry (i, i+offset) = bands[offset][i] (row-indexed)."""
    A = [[Fraction(0)] * n for _ in range(n)]
    for off, vals in bands.items():
        for i in range(n):
            j = i + off
            if 0 <= j < n:
                A[i][j] = Fraction(vals[i])
    return A


def exact_solve(A, b):
    """Gaussian elimination with row exchange on a zero pivot, in exact rationals."""
    n = len(A)
    M = [[Fraction(v) for v in row] + [Fraction(b[i])] for i, row in enumerate(A)]
    for k in range(n):
        p = next(r for r in range(k, n) if M[r][k] != 0)
        M[k], M[p] = M[p], M[k]
        for r in range(k + 1, n):
            if M[r][k] != 0:
                m = M[r][k] / M[k][k]
                for c in range(k, n + 1):
                    M[r][c] -= m * M[k][c]
    x = [Fraction(0)] * n
    for k in range(n - 1, -1, -1):
        x[k] = (M[k][n] - sum(M[k][c] * x[c] for c in range(k + 1, n))) / M[k][k]
    return x


def np_dense_from_bands(n, bands):
    A = np.zeros((n, n))
    for off, vals in bands.items():
        for i in range(n):
            j = i + off
            if 0 <= j < n:
                A[i, j] = vals[i]
    return A


def read_golden(path):
    """'key: v1 v2 ...' lines, values as rationals 'p/q' or decimals; '#' comments."""
    out = {}
    with open(path) as fh:
        for line in fh:
            line = line.split("#", 1)[0].strip()
            if not line:
                continue
            key, vals = line.split(":", 1)
            out[key.strip()] = [Fraction(v) for v in vals.split()]
    return out
