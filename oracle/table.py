"""Eq. 2 of the paper written out in numpy fp64 (ORACLE — test infrastructure, not the product).

PAPER.md §3.3: the truncation function T(x), x = r/2r_s, is tabulated on a grid of
nodes x_i over [0, 3] as two arrays,

    E_i = -4 exp(-x_i^2) / sqrt(pi),        T_i = erfc(x_i) - x_i E_i / 2,          (L143)

and evaluated at x = x_i + eps by the Taylor series (Eq. 2), term by term:

    T[0] = T_i
    T[1] = + x_i^2 E_i eps
    T[2] = - x_i (x_i^2 - 1) E_i eps^2
    T[3] = + (2/3 x_i^4 - 5/3 x_i^2 + 1/3) E_i eps^3
    T[4] = - x_i (1/3 x_i^4 - 3/2 x_i^2 + 1) E_i eps^4

``level`` k keeps T[0] .. T[k].  Readings (A14): nodes x_i = i*h, h = 3/n, i = 0..n
(n+1 entries so that the nearest node exists at x -> 3), nearest-node lookup (|eps| <= h/2).
The paper's own table has 512 nodes.

This follows the paper's notation on purpose; nothing here is shared with the CUDA table code.
Pins: tests/test_oracle_pins.py (error of level k scales as h^(k+1); T[k] equals the k-th Taylor
term of Eq. 1 obtained by finite differences / mpmath derivatives).
"""
from __future__ import annotations

import math

import numpy as np

X_MAX = 3.0   # table range in x = r/2r_s


def make_table(n: int):
    """(x_i, T_i, E_i) for i = 0..n in fp64."""
    # math.erfc per node keeps this independent of scipy
    x = np.arange(n + 1, dtype=np.float64) * (X_MAX / n)
    E = -4.0 * np.exp(-x * x) / math.sqrt(math.pi)
    T = np.array([math.erfc(v) for v in x]) - x * E / 2.0
    return x, T, E


def eval_table(xq, n: int, level: int, *, lookup: str = "nearest"):
    """Eq. 2 up to T[level] at the points xq (0 <= xq <= 3), fp64."""
    xq = np.asarray(xq, dtype=np.float64)
    x, T, E = make_table(n)
    h = X_MAX / n
    if lookup == "nearest":
        i = np.floor(xq / h + 0.5).astype(np.int64)
    elif lookup == "floor":
        i = np.floor(xq / h).astype(np.int64)
    else:
        raise ValueError(lookup)
    i = np.clip(i, 0, n)
    xi, Ti, Ei = x[i], T[i], E[i]
    eps = xq - xi
    terms = [
        Ti,
        xi ** 2 * Ei * eps,
        -xi * (xi ** 2 - 1.0) * Ei * eps ** 2,
        (2.0 / 3.0 * xi ** 4 - 5.0 / 3.0 * xi ** 2 + 1.0 / 3.0) * Ei * eps ** 3,
        -xi * (1.0 / 3.0 * xi ** 4 - 3.0 / 2.0 * xi ** 2 + 1.0) * Ei * eps ** 4,
    ]
    if not 0 <= level <= 4:
        raise ValueError("level must be 0..4")
    out = np.zeros_like(xq)
    for k in range(level + 1):
        out = out + terms[k]
    return out
