"""Pins for the truncated-M2L oracle (oracle/m2l.py): what PAPER.md §2 L41-L51 and the mathematics fix,
independent of the oracle's own code.  CPU only.

f_(n) (L51) against symbolic (1/r d/dr)^n psi; the inverse-square limit L45; D_n against symbolic partial derivatives
of psi; the trace of D_2 against the closed form of laplace(psi) (reading A24: not traceless); the whole chain
P2M -> M2L -> L2P against direct sums, with the error falling as (size / separation)^(p+1)."""
import math

import numpy as np
import pytest
import sympy as sp


@pytest.fixture(scope="module")
def m2l():
    from oracle import m2l as mod
    return mod


R_S = 0.31


def _psi_sym():
    r, rs = sp.symbols("r r_s", positive=True)
    return r, rs, sp.erfc(r / (2 * rs)) / r


@pytest.mark.parametrize("n", [0, 1, 2, 3, 4, 5, 6])
def test_prefactor_f_n_is_the_radial_derivative_operator(m2l, n):
    """L51's closed form == (1/r d/dr)^n [erfc(r/2r_s)/r], by symbolic differentiation evaluated to 40 digits."""
    r, rs, g = _psi_sym()
    for _ in range(n):
        g = sp.diff(g, r) / r
    for rv in (0.07, 0.4, 1.1, 1.86):           # x = r/2r_s from 0.11 to 3
        want = float(g.subs({r: sp.Float(rv, 40), rs: sp.Float(R_S, 40)}).evalf(40))
        got = float(m2l.f_n(n, np.array([rv]), R_S)[0])
        assert got == pytest.approx(want, rel=2e-11)


def test_prefactor_signs_and_inverse_square_limit(m2l):
    # f_(0) = psi itself; f_(1) = psi'/r = -T/r^3 (Eq. 1)
    rv = 0.5
    x = rv / (2 * R_S)
    T = math.erfc(x) + 2 * x / math.sqrt(math.pi) * math.exp(-x * x)
    assert m2l.f_n(0, [rv], R_S)[0] == pytest.approx(math.erfc(x) / rv, rel=1e-14)
    assert m2l.f_n(1, [rv], R_S)[0] == pytest.approx(-T / rv ** 3, rel=1e-14)
    # L45: r_s -> infinity recovers (-1)^n (2n-1)!! / r^(2n+1)
    for n in range(7):
        want = (-1) ** n * np.prod(np.arange(2 * n - 1, 0, -2)) / rv ** (2 * n + 1)
        assert m2l.f_n_inverse_square(n, [rv])[0] == pytest.approx(want, rel=1e-14)
        assert m2l.f_n(n, [rv], 1e5)[0] == pytest.approx(want, rel=1e-4)


def test_derivative_tensor_against_symbolic_partials(m2l):
    """D_n = d^n psi / dx^nx dy^ny dz^nz for every |n| <= 4 (35 components) and a few of order 5, 6."""
    x, y, z = sp.symbols("x y z", real=True)
    rs = sp.Float(R_S, 40)
    rr = sp.sqrt(x * x + y * y + z * z)
    psi = sp.erfc(rr / (2 * rs)) / rr
    R = np.array([[0.23, -0.41, 0.37]])
    at = {x: sp.Float(R[0, 0], 40), y: sp.Float(R[0, 1], 40), z: sp.Float(R[0, 2], 40)}
    D = m2l.derivative_tensors(R, 6, R_S)
    check = m2l.multi_indices(4) + [(5, 0, 0), (2, 2, 1), (0, 1, 4), (1, 1, 3), (2, 2, 2), (0, 6, 0), (3, 1, 2)]
    for n in check:
        expr = psi
        for var, k in zip((x, y, z), n):
            if k:
                expr = sp.diff(expr, var, k)
        want = float(expr.subs(at).evalf(40))
        assert float(D[n][0]) == pytest.approx(want, rel=1e-10, abs=1e-12), n


def test_trace_of_D2_is_the_screening_density_not_zero(m2l):
    """Reading A24: laplace(erfc(r/2r_s)/r) = exp(-r^2/4r_s^2) / (2 sqrt(pi) r_s^3), so D_n is not traceless for the
    truncated kernel; for psi = 1/r (L45) it is."""
    R = np.array([[0.3, 0.1, -0.25], [0.02, 0.5, 0.4]])
    r = np.sqrt((R * R).sum(axis=1))
    D = m2l.derivative_tensors(R, 4, R_S)
    tr = D[(2, 0, 0)] + D[(0, 2, 0)] + D[(0, 0, 2)]
    assert tr == pytest.approx(np.exp(-r * r / (4 * R_S ** 2)) / (2 * math.sqrt(math.pi) * R_S ** 3), rel=1e-12)
    # higher orders: grad^n of the same scalar identity, e.g. the trace over the last two indices of D_4
    tr4 = D[(2, 2, 0)] + D[(0, 4, 0)] + D[(0, 2, 2)]      # d^2/dy^2 of laplace(psi)
    lap = lambda yy: math.exp(-(R[0, 0] ** 2 + yy ** 2 + R[0, 2] ** 2) / (4 * R_S ** 2)) / (2 * math.sqrt(math.pi) * R_S ** 3)
    h = 1e-4
    num = (lap(R[0, 1] + h) - 2 * lap(R[0, 1]) + lap(R[0, 1] - h)) / h ** 2
    assert tr4[0] == pytest.approx(num, rel=1e-5)
    Dn = m2l.derivative_tensors(R, 4, R_S, newtonian=True)
    scale = np.abs(Dn[(2, 0, 0)])
    assert np.all(np.abs(Dn[(2, 0, 0)] + Dn[(0, 2, 0)] + Dn[(0, 0, 2)]) < 1e-13 * scale)


def _two_clusters(seed, size, sep, n_a=40, n_b=25):
    rng = np.random.default_rng(seed)
    zA = np.array([0.2, 0.3, 0.25])
    direction = np.array([0.6, -0.48, 0.64])
    zB = zA + sep * direction / np.linalg.norm(direction)
    ya = zA + size * (rng.random((n_a, 3)) - 0.5)
    ma = rng.uniform(0.5, 1.5, n_a)
    xb = zB + size * (rng.random((n_b, 3)) - 0.5)
    return zA, zB, ya, ma, xb


def _direct(ya, ma, xb, r_s, G=1.0):
    """phi(x) = -G sum m erfc(r/2r_s)/r and a(x) = G sum m T(r) (y - x)/r^3  (Eq. 1), plain loops."""
    phi = np.zeros(len(xb))
    acc = np.zeros((len(xb), 3))
    for i, xv in enumerate(xb):
        d = ya - xv
        r = np.sqrt((d * d).sum(axis=1))
        u = r / (2 * r_s)
        erfc = np.array([math.erfc(v) for v in u])
        T = erfc + 2 * u / math.sqrt(math.pi) * np.exp(-u * u)
        phi[i] = -G * (ma * erfc / r).sum()
        acc[i] = G * ((ma * T / r ** 3)[:, None] * d).sum(axis=0)
    return phi, acc


def test_p2m_m2l_l2p_converges_to_the_direct_sum(m2l):
    """The whole chain against the definition: error ~ (size/separation)^(p+1), geometric in p."""
    size, sep = 0.1, 0.6
    zA, zB, ya, ma, xb = _two_clusters(3, size, sep)
    phi_ref, acc_ref = _direct(ya, ma, xb, R_S, G=1.3)
    err_phi, err_acc = [], []
    for p in range(0, 8):
        M = m2l.p2m(ya, ma, zA, p)
        L = m2l.m2l(np.stack([zA, zB]), np.stack([M, np.zeros_like(M)]), [(1, 0)], p, R_S)
        phi, acc = m2l.l2p(L[1], zB, xb, p, G=1.3)
        err_phi.append(np.abs(phi - phi_ref).max() / np.abs(phi_ref).max())
        err_acc.append(np.abs(acc - acc_ref).max() / np.abs(acc_ref).max())
    assert err_phi[0] < 0.3 and err_phi[7] < 1e-6 and err_acc[7] < 2e-5
    for p in range(1, 8):                      # each order gains roughly the factor separation/size-ish
        assert err_phi[p] < 0.5 * err_phi[p - 1]
    # halving the cluster size at fixed p = 4 gains about 2^5
    zA2, zB2, ya2, ma2, xb2 = _two_clusters(3, size / 2, sep)
    phi_ref2, _ = _direct(ya2, ma2, xb2, R_S)
    M2 = m2l.p2m(ya2, ma2, zA2, 4)
    L2 = m2l.m2l(np.stack([zA2, zB2]), np.stack([M2, np.zeros_like(M2)]), [(1, 0)], 4, R_S)
    phi2, _ = m2l.l2p(L2[1], zB2, xb2, 4)
    zA1, zB1, ya1, ma1, xb1 = _two_clusters(3, size, sep)
    phi_ref1, _ = _direct(ya1, ma1, xb1, R_S)
    M1 = m2l.p2m(ya1, ma1, zA1, 4)
    L1 = m2l.m2l(np.stack([zA1, zB1]), np.stack([M1, np.zeros_like(M1)]), [(1, 0)], 4, R_S)
    phi1, _ = m2l.l2p(L1[1], zB1, xb1, 4)
    gain = np.abs(phi1 - phi_ref1).max() / np.abs(phi2 - phi_ref2).max()
    assert 12 < gain < 90


def test_m2l_of_a_point_mass_is_m_times_D_and_lists_add_up(m2l):
    p = 4
    idx = {n: c for c, n in enumerate(m2l.multi_indices(p))}
    centres = np.array([[0.1, 0.2, 0.3], [0.7, 0.1, 0.5], [0.4, 0.9, 0.2]])
    M = np.zeros((3, m2l.n_coeffs(p)))
    M[0, 0] = 2.5                                  # a point mass at the centre of cell 0: only M_0
    L = m2l.m2l(centres, M, [(1, 0)], p, R_S)
    D = m2l.derivative_tensors((centres[1] - centres[0])[None, :], p, R_S)
    for n, c in idx.items():
        assert L[1, c] == pytest.approx(2.5 * D[n][0], rel=1e-14, abs=1e-300)
    assert np.all(L[0] == 0) and np.all(L[2] == 0)
    # two sources into one target = sum of the two single-pair results; a dipole-only source uses D_{n+e_x}
    M[2, idx[(1, 0, 0)]] = -0.75
    both = m2l.m2l(centres, M, [(1, 0), (1, 2)], p, R_S)
    one = m2l.m2l(centres, M, [(1, 2)], p, R_S)
    assert both[1] == pytest.approx(L[1] + one[1], rel=1e-14)
    D2 = m2l.derivative_tensors((centres[1] - centres[2])[None, :], p, R_S)
    assert one[1, idx[(0, 1, 0)]] == pytest.approx(-0.75 * D2[(1, 1, 0)][0], rel=1e-14)
    assert one[1, idx[(4, 0, 0)]] == 0.0           # |n| = p leaves only m = 0, and M_0 of cell 2 is zero


def test_m2l_periodic_image_shift(m2l):
    p = 3
    centres = np.array([[0.95, 0.5, 0.5], [0.05, 0.5, 0.5]])
    M = np.zeros((2, m2l.n_coeffs(p)))
    M[0] = np.arange(1, m2l.n_coeffs(p) + 1) * 0.1
    # source cell 0 seen from target cell 1 through the seam: source moved by -1 box length along x
    a = m2l.m2l(centres, M, [(1, 0)], p, R_S, boxsize=1.0, shifts=[(-1, 0, 0)])
    moved = centres.copy()
    moved[0, 0] -= 1.0
    b = m2l.m2l(moved, M, [(1, 0)], p, R_S)
    assert np.array_equal(a, b)
    assert m2l.n_coeffs(3) == 20 and m2l.n_coeffs(4) == 35 and len(m2l.multi_indices(6)) == 84
