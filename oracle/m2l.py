"""Truncated M2L in numpy fp64 (ORACLE — test infrastructure, not the product).

PAPER.md §2 L41-L51.  The short-range potential of a unit mass is  psi(r) = erfc(r / 2 r_s) / r  (the potential
whose force is Eq. 1: psi'(r) = -T(r; r_s) / r^2, L55-L59), and the multipole-to-local operator is (L41)

    L_n(z_B) = sum_{|m| = 0}^{p - |n|}  M_m(z_A)  D_{n+m}(z_B - z_A),          D_n = grad^n psi(r)            (L41-L43)

with multi-indices n = (n_x, n_y, n_z).  The radial derivatives that build D_n are the paper's prefactors (L51)

    (-1)^n r_s^(2n+1) f_(n)(x) = (2n-1)!!/2^(2n+1) erfc(x)/x^(2n+1)
                                 + sum_{q=1}^{n} 2^(-q-n) (2n-1)!!/(2n-2q+1)!!  exp(-x^2)/(sqrt(pi) x^(2q)),   x = r/2r_s,

i.e. f_(n)(r) = (1/r d/dr)^n psi(r)  (checked against symbolic derivatives in tests/test_m2l_oracle.py; for the
inverse-square law they reduce to L45, f_(n)^inv = (-1)^n (2n-1)!!/r^(2n+1)).

Readings (A24-A26; the paper defers every detail to Wang 2021, which is not available):
  A24  D_n is the full Cartesian derivative tensor of psi.  The paper writes D_n = f_(n) r^n "traceless", which is exact
       only for a harmonic kernel: for the truncated psi, laplace(psi) = exp(-x^2) / (2 sqrt(pi) r_s^3) != 0, so the
       trace terms are kept.  D_n is assembled from the f_(k) by the radial-derivative recursion
           D^(k)_0 = f_(k),   D^(k)_{n + e_i} = R_i D^(k+1)_n + n_i D^(k+1)_{n - e_i},   D_n = D^(0)_n.
  A25  Multipoles about the source centre carry the Taylor factors:  M_m(z_A) = sum_j m_j (-a_j)^m / m!,
       a_j = y_j - z_A;  then  sum_j m_j psi(x - y_j) ~= sum_{|n| <= p} L_n(z_B) b^n / n!,  b = x - z_B,
       the potential is -G times that and the acceleration +G times its gradient.
  A26  The expansion order p and the cell-pair list are inputs (the paper gives neither).  A pair may carry a
       periodic image shift s in {-1,0,+1}^3 box lengths added to the source centre.

Nothing here is shared with the CUDA path.
"""
from __future__ import annotations

import math

import numpy as np


def multi_indices(p: int):
    """All (n_x, n_y, n_z) with |n| <= p, ordered by |n|, then n_x descending, then n_y descending."""
    out = []
    for k in range(p + 1):
        for nx in range(k, -1, -1):
            for ny in range(k - nx, -1, -1):
                out.append((nx, ny, k - nx - ny))
    return out


def n_coeffs(p: int) -> int:
    return (p + 1) * (p + 2) * (p + 3) // 6


def _dfact(k: int) -> int:
    """(k)!! for odd k >= -1, with (-1)!! = 1."""
    out = 1
    while k > 1:
        out *= k
        k -= 2
    return out


def f_n(n: int, r, r_s: float):
    """The paper's prefactor f_(n) (L51), written term by term.  r: array of separations > 0."""
    r = np.asarray(r, dtype=np.float64)
    x = r / (2.0 * r_s)
    erfc = np.vectorize(math.erfc)(x)
    val = _dfact(2 * n - 1) / 2.0 ** (2 * n + 1) * erfc / x ** (2 * n + 1)
    for q in range(1, n + 1):
        val = val + 2.0 ** (-q - n) * _dfact(2 * n - 1) / _dfact(2 * n - 2 * q + 1) * np.exp(-x * x) / (math.sqrt(math.pi) * x ** (2 * q))
    return (-1.0) ** n * val / r_s ** (2 * n + 1)


def f_n_inverse_square(n: int, r):
    """L45: the prefactor of the plain inverse-square law."""
    return (-1.0) ** n * _dfact(2 * n - 1) / np.asarray(r, dtype=np.float64) ** (2 * n + 1)


def derivative_tensors(R, p: int, r_s: float, *, newtonian: bool = False):
    """D_n(R) = grad^n psi at the separations R[npairs, 3], for all |n| <= p (reading A24).
    Returns {n: array[npairs]}.  newtonian=True uses psi = 1/r (L45) instead."""
    R = np.atleast_2d(np.asarray(R, dtype=np.float64))
    r = np.sqrt((R * R).sum(axis=1))
    f = [f_n_inverse_square(k, r) if newtonian else f_n(k, r, r_s) for k in range(p + 1)]
    # level[k][n] = D^(k)_n for |n| <= p - k
    level = [dict() for _ in range(p + 1)]
    for k in range(p + 1):
        level[k][(0, 0, 0)] = f[k]
    for order in range(1, p + 1):
        for k in range(p - order + 1):
            for n in (m for m in multi_indices(order) if sum(m) == order):
                i = 0 if n[0] > 0 else (1 if n[1] > 0 else 2)          # lower n along its first non-zero axis
                base = list(n)
                base[i] -= 1
                val = R[:, i] * level[k + 1][tuple(base)]
                if base[i] > 0:
                    low = list(base)
                    low[i] -= 1
                    val = val + base[i] * level[k + 1][tuple(low)]
                level[k][n] = val
    return level[0]


def p2m(pos, mass, centre, p: int):
    """M_m(z_A) = sum_j m_j (-a_j)^m / m!  (reading A25).  Returns array[n_coeffs(p)] in multi_indices order."""
    a = np.asarray(pos, dtype=np.float64) - np.asarray(centre, dtype=np.float64)
    mass = np.asarray(mass, dtype=np.float64)
    out = np.empty(n_coeffs(p))
    for c, (mx, my, mz) in enumerate(multi_indices(p)):
        w = (-a[:, 0]) ** mx * (-a[:, 1]) ** my * (-a[:, 2]) ** mz
        out[c] = (mass * w).sum() / (math.factorial(mx) * math.factorial(my) * math.factorial(mz))
    return out


def m2l(centres, multipoles, pairs, p: int, r_s: float, *, boxsize: float = 0.0, shifts=None, newtonian: bool = False):
    """L_n(z_B) = sum over listed pairs (B, A) of sum_{|m| <= p - |n|} M_m(z_A) D_{n+m}(z_B - z_A)   (L41).

    centres[n_cells, 3]; multipoles[n_cells, n_coeffs(p)]; pairs[n_pairs, 2] = (target cell B, source cell A);
    shifts[n_pairs, 3] in {-1, 0, +1} box lengths added to the source centre (A26), or None.
    Returns locals[n_cells, n_coeffs(p)]."""
    centres = np.asarray(centres, dtype=np.float64)
    multipoles = np.asarray(multipoles, dtype=np.float64)
    pairs = np.asarray(pairs, dtype=np.int64).reshape(-1, 2)
    idx = {n: c for c, n in enumerate(multi_indices(p))}
    src = centres[pairs[:, 1]]
    if shifts is not None:
        src = src + boxsize * np.asarray(shifts, dtype=np.float64)
    R = centres[pairs[:, 0]] - src
    D = derivative_tensors(R, p, r_s, newtonian=newtonian)
    contrib = np.zeros((len(pairs), n_coeffs(p)))
    for n in multi_indices(p):
        for m in multi_indices(p - sum(n)):
            nm = (n[0] + m[0], n[1] + m[1], n[2] + m[2])
            contrib[:, idx[n]] += multipoles[pairs[:, 1], idx[m]] * D[nm]
    out = np.zeros((len(centres), n_coeffs(p)))
    np.add.at(out, pairs[:, 0], contrib)
    return out


def l2p(local, centre, x, p: int, G: float = 1.0):
    """Potential and acceleration at the points x[npts, 3] from the local expansion about `centre` (A25):
    psi_sum = sum_n L_n b^n / n!,  phi = -G psi_sum,  a = +G grad psi_sum."""
    b = np.atleast_2d(np.asarray(x, dtype=np.float64)) - np.asarray(centre, dtype=np.float64)
    psi = np.zeros(len(b))
    grad = np.zeros((len(b), 3))
    for c, n in enumerate(multi_indices(p)):
        fact = math.factorial(n[0]) * math.factorial(n[1]) * math.factorial(n[2])
        psi += local[c] * b[:, 0] ** n[0] * b[:, 1] ** n[1] * b[:, 2] ** n[2] / fact
        for i in range(3):
            if n[i] == 0:
                continue
            e = list(n)
            e[i] -= 1
            fe = math.factorial(e[0]) * math.factorial(e[1]) * math.factorial(e[2])
            grad[:, i] += local[c] * b[:, 0] ** e[0] * b[:, 1] ** e[1] * b[:, 2] ** e[2] / fe
    return -G * psi, G * grad
