"""Pins for the CPU oracle (oracle/): what the paper and the mathematics fix, independent of the
oracle's own code.  CPU only.

Citations: PAPER.md L55-L59 (force form, Eq. 1), L125 (integral form of T), L129-L143 (Eq. 2 and the
table), L33 (Gaussian split, r_s = 1.2 BOXSIZE/N_PM), L53 (x = r/2r_s, cut-off); DESIGN.md readings
A1-A14.
"""
import math
import os

import mpmath
import numpy as np
import pytest
from scipy import integrate

from paper_2107_14008_b200 import workloads

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
SQRT_PI = math.sqrt(math.pi)


def _golden(name):
    out = {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.strip()
            if line and not line.startswith("#"):
                k, v = line.split()
                out[k] = float(v)
    return out


def T_mp(x):
    """Eq. 1 in 40-digit mpmath: an evaluation that shares nothing with libm or the oracle."""
    with mpmath.workdps(40):
        x = mpmath.mpf(x)
        return mpmath.erfc(x) + 2 * x / mpmath.sqrt(mpmath.pi) * mpmath.exp(-x * x)


# ----------------------------------------------------------------------------- g / T (Eq. 1)

@pytest.mark.parametrize("x", [0.0, 1e-3, 0.1, 0.5, 1.0, 1.7, 2.0, 2.5, 3.0, 4.0])
def test_T_closed_form_vs_mpmath(oracle, x):
    assert oracle.oracle_T(x) == pytest.approx(float(T_mp(x)), rel=2e-14, abs=1e-18)


@pytest.mark.parametrize("x", [0.0, 0.05, 0.3, 1.0, 2.0, 3.0])
def test_T_integral_form_L125(oracle, x):
    # T(x) = 4/sqrt(pi) * int_x^inf u^2 exp(-u^2) du
    val, err = integrate.quad(lambda u: u * u * math.exp(-u * u), x, np.inf, epsabs=1e-14, epsrel=1e-13)
    assert oracle.oracle_T(x) == pytest.approx(4.0 / SQRT_PI * val, rel=1e-12, abs=1e-14)


def test_T_derivative_from_integral_form(oracle):
    # dT/dx = -(4/sqrt(pi)) x^2 exp(-x^2), by central differences of the oracle's T
    for x in [0.2, 0.9, 1.5, 2.6]:
        h = 1e-5
        num = (oracle.oracle_T(x + h) - oracle.oracle_T(x - h)) / (2 * h)
        assert num == pytest.approx(-4.0 / SQRT_PI * x * x * math.exp(-x * x), rel=1e-8)


def test_T_newtonian_limit_series(oracle):
    # g -> 1 as r/r_s -> 0 (north_star); leading deviation -4 x^3 / (3 sqrt(pi)) from L125
    assert oracle.oracle_T(0.0) == 1.0
    for x in [1e-4, 1e-3, 1e-2]:
        series = 1.0 - 4 * x ** 3 / (3 * SQRT_PI) + 4 * x ** 5 / (5 * SQRT_PI) - 2 * x ** 7 / (7 * SQRT_PI)
        assert oracle.oracle_T(x) == pytest.approx(series, abs=1e-15 + x ** 9)
    xs = np.linspace(0, 3.5, 200)
    Ts = oracle.oracle_T(xs)
    assert np.all(np.diff(Ts) < 0) and Ts[-1] > 0          # monotone decreasing, positive


def test_T_at_cut_value(oracle):
    # value of the jump at r_cut = 6 r_s, x = 3 (A1)
    assert oracle.oracle_T(3.0) == pytest.approx(4.39849652838829e-4, rel=1e-12)
    assert float(T_mp(3)) == pytest.approx(4.39849652838829e-4, rel=1e-13)


@pytest.mark.parametrize("r_over_rs", [0.05, 0.5, 1.0, 2.5, 5.0, 6.0])
def test_split_identity_with_long_range_fourier(oracle, r_over_rs):
    """g * (long-range Gaussian complement) reproduces 1/r^2 (north_star).

    The long-range pair-force factor is derived from the Fourier-space Green function
    exp(-k^2 r_s^2)/k^2 (A2), independently of Eq. 1:
        g_long(r) = (2/pi) int_0^inf exp(-k^2 r_s^2) [sin(kr)/k - r cos(kr)] dk
    and g + g_long must equal 1.
    """
    r_s = 0.0375
    r = r_over_rs * r_s

    def integrand(k):
        if k == 0.0:
            return 0.0
        return math.exp(-k * k * r_s * r_s) * (math.sin(k * r) / k - r * math.cos(k * r))

    val, err = integrate.quad(integrand, 0.0, 12.0 / r_s, limit=2000, epsabs=1e-16, epsrel=1e-13)
    g_long = 2.0 / math.pi * val
    g = oracle.oracle_T(r / (2 * r_s))
    assert g + g_long == pytest.approx(1.0, abs=5e-12)


# ----------------------------------------------------------------------------- two-body closed forms

def _two_body(oracle, p1, p2, m=(0.3, 0.7), L=1.0, n_pm=32, G=1.0):
    r_s = 1.2 * L / n_pm
    pos = np.array([p1, p2], dtype=np.float64)
    mass = np.array(m, dtype=np.float64)
    acc, cnt = oracle.p2p(pos, mass, boxsize=L, r_s=r_s, r_cut=6 * r_s, G=G)
    return acc, cnt, r_s


def test_two_body_on_axis(oracle):
    d = 0.05
    acc, cnt, r_s = _two_body(oracle, [0.2, 0.5, 0.5], [0.2 + d, 0.5, 0.5])
    g = float(T_mp(d / (2 * r_s)))
    # particle 0 is pulled towards particle 1 (+x) with G m_2 g / d^2      (L55, Alg. 2 sign)
    assert acc[0, 0] == pytest.approx(0.7 * g / d ** 2, rel=1e-13)
    assert acc[1, 0] == pytest.approx(-0.3 * g / d ** 2, rel=1e-13)
    assert np.all(acc[:, 1:] == 0.0)
    assert cnt == {"pair_tests": 4, "pairs_in_cut": 2}


def test_two_body_across_periodic_seam(oracle):
    d = 0.03
    acc, cnt, r_s = _two_body(oracle, [0.99, 0.5, 0.01], [0.99 + d - 1.0, 0.5, 0.01 - d + 1.0])
    # separation vector (min image) = (+d, 0, -d)
    r = d * math.sqrt(2)
    f = 0.7 * float(T_mp(r / (2 * r_s))) / r ** 3
    assert acc[0] == pytest.approx([f * d, 0.0, -f * d], rel=1e-12, abs=1e-15)


def test_two_body_general_direction_and_G(oracle):
    dvec = np.array([0.011, -0.027, 0.033])
    p1 = np.array([0.4, 0.6, 0.1])
    acc, cnt, r_s = _two_body(oracle, p1, p1 + dvec, G=2.5)
    r = float(np.linalg.norm(dvec))
    f = 2.5 * 0.7 * float(T_mp(r / (2 * r_s))) / r ** 3
    assert acc[0] == pytest.approx(f * dvec, rel=1e-12)
    assert 0.3 * acc[0] + 0.7 * acc[1] == pytest.approx([0, 0, 0], abs=1e-14 * abs(f) * r)


def test_zero_beyond_cut_and_jump_at_cut(oracle):
    L, n_pm = 1.0, 32
    r_s = 1.2 * L / n_pm
    r_cut = 6 * r_s
    for d, expect_zero in [(r_cut, True), (r_cut * (1 + 1e-12), True), (0.3, True), (0.49, True),
                           (r_cut * (1 - 1e-9), False)]:
        acc, cnt, _ = _two_body(oracle, [0.0, 0.1, 0.1], [d, 0.1, 0.1], m=(1.0, 1.0))   # dx == d exactly
        if expect_zero:
            assert np.all(acc == 0.0) and cnt["pairs_in_cut"] == 0
        else:
            assert acc[0, 0] == pytest.approx(4.39849652838829e-4 / r_cut ** 2, rel=1e-7)


def test_coincident_particles_contribute_nothing(oracle):
    acc, cnt, _ = _two_body(oracle, [0.3, 0.3, 0.3], [0.3, 0.3, 0.3])
    assert np.all(acc == 0.0) and cnt["pairs_in_cut"] == 0


# ----------------------------------------------------------------------------- sums

@pytest.fixture(scope="module")
def small_uniform():
    cfg = workloads.scaled(1, 16)          # 4096 particles, N_PM = 16
    pos, mass = workloads.make(cfg)
    r_s = 1.2 * cfg.boxsize / cfg.n_pm
    return cfg, pos, mass, r_s


def test_newtons_third_law(oracle, small_uniform):
    cfg, pos, mass, r_s = small_uniform
    rng = np.random.default_rng(5)
    mass = mass * rng.uniform(0.5, 2.0, size=mass.shape)       # unequal masses make this sharper
    acc, _ = oracle.p2p(pos, mass, boxsize=1.0, r_s=r_s, r_cut=6 * r_s)
    num = np.linalg.norm((mass[:, None] * acc).sum(axis=0))
    den = (mass * np.linalg.norm(acc, axis=1)).sum()
    assert num / den < 1e-12            # north_star: total momentum change < 1e-12 relative


def test_mean_neighbour_count_closed_form(oracle, small_uniform):
    # homogeneous input with N = N_PM^3: <neighbours inside r_cut> = 4 pi/3 * 7.2^3 = 1563.5
    cfg, pos, mass, r_s = small_uniform
    _, cnt = oracle.p2p(pos, mass, boxsize=1.0, r_s=r_s, r_cut=6 * r_s)
    assert cnt["pair_tests"] == cfg.n ** 2
    mean = cnt["pairs_in_cut"] / cfg.n
    assert mean == pytest.approx(4 * math.pi / 3 * 7.2 ** 3, rel=0.01)


def test_perfect_lattice_has_zero_force(oracle):
    side = 16              # r_cut = 7.2/16 < L/2, as minimum image requires (A10)
    g = (np.arange(side) + 0.5) / side
    pos = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3)
    mass = np.full(len(pos), 1.0 / len(pos))
    r_s = 1.2 / side
    acc, cnt = oracle.p2p(pos, mass, boxsize=1.0, r_s=r_s, r_cut=6 * r_s)
    scale = mass[0] / (1.0 / side) ** 2          # one neighbour at one grid spacing
    assert cnt["pairs_in_cut"] > 0
    assert np.abs(acc).max() < 1e-12 * scale


def test_translation_and_axis_covariance(oracle):
    cfg = workloads.scaled(1, 8)
    pos, mass = workloads.make(cfg, flavour="D")
    r_s = 1.2 / cfg.n_pm
    kw = dict(boxsize=1.0, r_s=r_s, r_cut=6 * r_s)
    a0, _ = oracle.p2p(pos, mass, **kw)
    rms = np.sqrt((a0 ** 2).sum(axis=1).mean())
    # rigid translation mod L (positions stay on a common 2^-20 grid so the shift is exact)
    q = np.round(pos * 2 ** 20) / 2 ** 20
    a_q, _ = oracle.p2p(q, mass, **kw)
    shift = np.array([0.25, 0.5, 0.8125])
    a_s, _ = oracle.p2p(np.mod(q + shift, 1.0), mass, **kw)
    assert np.abs(a_s - a_q).max() < 1e-12 * rms
    # axis permutation and reflection
    a_p, _ = oracle.p2p(np.ascontiguousarray(pos[:, [2, 0, 1]]), mass, **kw)
    assert np.abs(a_p - a0[:, [2, 0, 1]]).max() < 1e-13 * rms
    refl = np.mod(-q, 1.0)
    a_r, _ = oracle.p2p(refl, mass, **kw)
    assert np.abs(a_r + a_q).max() < 1e-12 * rms


@pytest.mark.parametrize("n", [2, 3, 8, 64])
def test_tiny_n_brute_force_mpmath(oracle, n):
    """Independent 40-digit evaluation of the definition on tiny inputs."""
    rng = np.random.default_rng(100 + n)
    L, n_pm, G = 1.0, 16, 1.0
    r_s = 1.2 * L / n_pm
    r_cut = 6 * r_s
    pos = rng.random((n, 3)) * 0.6 + 0.7        # straddles the periodic seam after wrapping
    pos = np.mod(pos, 1.0)
    mass = rng.uniform(0.5, 1.5, n)
    acc, _ = oracle.p2p(pos, mass, boxsize=L, r_s=r_s, r_cut=r_cut, G=G)
    with mpmath.workdps(40):
        ref = np.zeros((n, 3))
        for i in range(n):
            a = [mpmath.mpf(0)] * 3
            for j in range(n):
                d = [mpmath.mpf(pos[j, k]) - mpmath.mpf(pos[i, k]) for k in range(3)]
                d = [dk - L * mpmath.nint(dk / L) for dk in d]
                r2 = sum(dk * dk for dk in d)
                if r2 > 0 and r2 < mpmath.mpf(r_cut) ** 2:
                    r = mpmath.sqrt(r2)
                    x = r / (2 * mpmath.mpf(r_s))
                    T = mpmath.erfc(x) + 2 * x / mpmath.sqrt(mpmath.pi) * mpmath.exp(-x * x)
                    w = G * mpmath.mpf(mass[j]) * T / r ** 3
                    a = [a[k] + w * d[k] for k in range(3)]
            ref[i] = [float(v) for v in a]
    scale = np.abs(ref).max() if np.abs(ref).max() > 0 else 1.0
    assert np.abs(acc - ref).max() <= 1e-14 * scale


def test_sampled_mode_equals_full_mode_bitwise(oracle, small_uniform):
    cfg, pos, mass, r_s = small_uniform
    full, _ = oracle.p2p(pos, mass, boxsize=1.0, r_s=r_s, r_cut=6 * r_s)
    tgt = workloads.sample_targets(cfg.n, 257, cfg.seed)
    samp, cnt = oracle.p2p_sampled(pos, mass, tgt, boxsize=1.0, r_s=r_s, r_cut=6 * r_s)
    assert np.array_equal(samp, full[tgt])
    assert cnt["pair_tests"] == 257 * cfg.n


# ----------------------------------------------------------------------------- Eq. 2 table

def test_table_matches_paper_parameters(oracle):
    g = _golden("paper_L143_table.txt")
    x, T, E = oracle.make_table(int(g["nodes"]))
    assert x[0] == g["x_min"] and x[-1] == g["x_max"] and len(x) == int(g["nodes"]) + 1
    # E_i and T_i as defined at L143, against mpmath
    for i in [0, 1, 100, 256, 511, 512]:
        with mpmath.workdps(30):
            xi = mpmath.mpf(x[i])
            Ei = -4 * mpmath.exp(-xi * xi) / mpmath.sqrt(mpmath.pi)
            Ti = mpmath.erfc(xi) - xi * Ei / 2
        assert E[i] == pytest.approx(float(Ei), rel=1e-14)
        assert T[i] == pytest.approx(float(Ti), rel=1e-13)
        assert T[i] == pytest.approx(float(T_mp(x[i])), rel=1e-13)      # T_i is Eq. 1 at the node


@pytest.mark.parametrize("level", [0, 1, 2, 3, 4])
def test_table_terms_are_taylor_coefficients(oracle, level):
    """T[k] of Eq. 2 must be T^(k)(x_i) eps^k / k! — checked against mpmath derivatives of Eq. 1."""
    n = 64
    h = 3.0 / n
    for i in [3, 17, 40, 60]:
        xi = i * h
        eps = 0.37 * h
        with mpmath.workdps(40):
            f = lambda t: mpmath.erfc(t) + 2 * t / mpmath.sqrt(mpmath.pi) * mpmath.exp(-t * t)
            want = sum(mpmath.diff(f, xi, k) * mpmath.mpf(eps) ** k / mpmath.factorial(k)
                       for k in range(level + 1))
        got = oracle.eval_table(np.array([xi + eps]), n, level)[0]
        assert got == pytest.approx(float(want), rel=1e-11, abs=1e-15)


def test_table_error_scales_as_h_to_level_plus_one(oracle):
    """Level-k error ~ h^(k+1) (Taylor remainder); orders of magnitude of Fig. 2 (L147-L149)."""
    xq = np.linspace(0.0, 3.0, 20001)
    exact = oracle.oracle_T(xq)
    err = {}
    for n in (256, 512, 1024):
        for level in range(5):
            approx = oracle.eval_table(xq, n, level)
            err[n, level] = np.max(np.abs(approx - exact) / exact)
    for level in range(4):                       # level 4 at n=1024 sits on fp64 round-off
        ratio = err[256, level] / err[512, level]
        assert 2 ** (level + 1) * 0.7 < ratio < 2 ** (level + 1) * 1.4
        assert err[512, level + 1] < err[512, level] * 0.05
    g = _golden("paper_L143_table.txt")
    n = int(g["nodes"])
    # "T[2] adequate for single precision": relative error of T at the fp32-epsilon scale or below 1e-6
    assert err[n, int(g["level_single"])] < 1e-6
    # "T[4] for double precision": far below T[2]; about 5e-12 for 512 nearest-node lookup
    assert err[n, int(g["level_double"])] < 1e-10
    # floor-node lookup is 2^(k+1) times worse than nearest-node lookup (A14)
    e_floor = np.max(np.abs(oracle.eval_table(xq, 512, 2, lookup="floor") - exact) / exact)
    assert 5.0 < e_floor / err[512, 2] < 11.0


# ----------------------------------------------------------------------------- paper's accounting

def test_paper_perf_accounting_is_self_consistent():
    g = _golden("paper_L218_perf_accounting.txt")
    peak = g["interactions_per_step"] * g["ops_per_interaction"] / g["kernel_seconds"] / 1e12
    avg = g["interactions_per_step"] * g["ops_per_interaction"] / g["step_seconds"] / 1e12
    assert peak == pytest.approx(g["peak_tflops_printed"], rel=2e-3)
    assert avg == pytest.approx(g["average_tflops_printed"], rel=2e-3)
    assert avg / g["machine_peak_tflops"] == pytest.approx(g["average_fraction_printed"], abs=0.01)
    # printed 48 %; plain arithmetic gives 49.3 % (A17)
    assert peak / g["machine_peak_tflops"] == pytest.approx(0.493, abs=0.002)


# ------------------------------------------------------------- isolated boundaries

def test_isolated_two_body_has_no_image_force(oracle):
    # across the seam of the unit box the periodic pair is close, the isolated pair is far beyond the cut
    n_pm = 32
    r_s = 1.2 / n_pm
    pos = np.array([[0.99, 0.5, 0.5], [0.02, 0.5, 0.5]])
    mass = np.array([1.0, 2.0])
    per, _ = oracle.p2p(pos, mass, boxsize=1.0, r_s=r_s, r_cut=6 * r_s)
    iso, cnt = oracle.p2p(pos, mass, boxsize=0.0, r_s=r_s, r_cut=6 * r_s)
    assert per[0, 0] > 0 and np.all(iso == 0.0) and cnt["pairs_in_cut"] == 0
    # a close isolated pair, negative coordinates allowed: closed form
    d = 0.04
    pos = np.array([[-0.3, 0.1, -2.0], [-0.3 + d, 0.1, -2.0]])
    iso, _ = oracle.p2p(pos, mass, boxsize=0.0, r_s=r_s, r_cut=6 * r_s)
    g = float(T_mp(d / (2 * r_s)))
    assert iso[0, 0] == pytest.approx(2.0 * g / d ** 2, rel=1e-13)
    assert iso[1, 0] == pytest.approx(-1.0 * g / d ** 2, rel=1e-13)


def test_isolated_equals_periodic_far_from_the_faces(oracle):
    # a blob that stays more than r_cut away from every face of the box feels no images: both modes agree bitwise
    rng = np.random.default_rng(11)
    n_pm = 32
    r_s = 1.2 / n_pm
    pos = 0.35 + 0.3 * rng.random((400, 3))
    mass = rng.uniform(0.5, 1.5, 400)
    per, c1 = oracle.p2p(pos, mass, boxsize=1.0, r_s=r_s, r_cut=6 * r_s)
    iso, c2 = oracle.p2p(pos, mass, boxsize=0.0, r_s=r_s, r_cut=6 * r_s)
    assert np.array_equal(per, iso) and c1 == c2
    # and Newton's third law holds in the isolated mode too
    tot = (mass[:, None] * iso).sum(axis=0)
    assert np.abs(tot).max() <= 1e-12 * (mass[:, None] * np.abs(iso)).sum()


# ---------------------------------------- Plummer softening (reading A23)

def _psi_mp(r, r_s):
    """Short-range potential of a unit mass, psi(r) = erfc(r/2r_s)/r (D_n = grad^n psi)."""
    return mpmath.erfc(r / (2 * r_s)) / r


def test_softening_zero_is_the_unsoftened_sum_bitwise(oracle, small_uniform):
    cfg, pos, mass, r_s = small_uniform
    kw = dict(boxsize=1.0, r_s=r_s, r_cut=6 * r_s)
    a0, c0 = oracle.p2p(pos, mass, **kw)
    a1, c1 = oracle.p2p(pos, mass, eps=0.0, **kw)
    a2, c2 = oracle.p2p(pos, mass, eps=1e-200, **kw)        # eps^2 underflows to 0
    assert np.array_equal(a0, a1) and np.array_equal(a0, a2) and c0 == c1 == c2
    # and a softening far below every pair separation changes the sum only at round-off level
    a3, _ = oracle.p2p(pos, mass, eps=1e-9, **kw)
    rms = np.sqrt((a0 ** 2).sum(axis=1).mean())
    assert np.abs(a3 - a0).max() < 1e-9 * rms


@pytest.mark.parametrize("eps_over_d", [0.01, 0.5, 1.0, 3.0, 40.0])
def test_softened_two_body_is_minus_gradient_of_plummer_substituted_potential(oracle, eps_over_d):
    """A23: a_1 = -grad_1 [ -G m_2 psi( sqrt(|r_1 - r_2|^2 + eps^2) ) ], by 40-digit numerical differentiation —
    fixes the direction vector (the unsoftened d), the radius in T and in 1/r^3 (both r_eps) and the sign."""
    n_pm, G = 32, 1.7
    r_s = 1.2 / n_pm
    dvec = np.array([0.004, -0.003, 0.0012])
    eps = eps_over_d * float(np.linalg.norm(dvec))
    if np.hypot(np.linalg.norm(dvec), eps) >= 6 * r_s:
        pytest.skip("beyond the cut")
    p1 = np.array([0.31, 0.52, 0.77])
    pos = np.array([p1, p1 + dvec])
    mass = np.array([0.4, 0.9])
    acc, cnt = oracle.p2p(pos, mass, boxsize=1.0, r_s=r_s, r_cut=6 * r_s, G=G, eps=eps)
    assert cnt["pairs_in_cut"] == 2
    with mpmath.workdps(40):
        def phi(x, y, z):      # potential at particle 1's position due to particle 2
            d2 = (pos[1, 0] - x) ** 2 + (pos[1, 1] - y) ** 2 + (pos[1, 2] - z) ** 2
            return -G * mass[1] * _psi_mp(mpmath.sqrt(d2 + mpmath.mpf(eps) ** 2), mpmath.mpf(r_s))
        want = [-mpmath.diff(phi, tuple(p1), tuple(int(k == a) for k in range(3))) for a in range(3)]
    assert acc[0] == pytest.approx([float(v) for v in want], rel=1e-11)
    assert 0.4 * acc[0] + 0.9 * acc[1] == pytest.approx([0, 0, 0], abs=1e-13 * np.abs(acc).max())


def test_softened_closed_form_limits_and_cut(oracle):
    n_pm = 32
    r_s = 1.2 / n_pm
    r_cut = 6 * r_s
    d, eps = 0.01, 0.02
    pos = np.array([[0.5, 0.5, 0.5], [0.5 + d, 0.5, 0.5]])
    mass = np.array([1.0, 2.0])
    acc, _ = oracle.p2p(pos, mass, boxsize=1.0, r_s=r_s, r_cut=r_cut, eps=eps)
    re = math.hypot(d, eps)
    assert acc[0, 0] == pytest.approx(2.0 * float(T_mp(re / (2 * r_s))) * d / re ** 3, rel=1e-13)
    # deep inside the softening core the force is linear in d: a -> G m d T(eps)/eps^3
    tiny = 1e-7
    pos[1, 0] = 0.5 + tiny
    acc, _ = oracle.p2p(pos, mass, boxsize=1.0, r_s=r_s, r_cut=r_cut, eps=eps)
    assert acc[0, 0] == pytest.approx(2.0 * float(T_mp(eps / (2 * r_s))) * tiny / eps ** 3, rel=1e-9)
    # coincident particles still contribute nothing (d = 0), and the cut acts on r_eps: a pair with
    # r < r_cut <= r_eps is outside
    pos[1] = pos[0]
    acc, cnt = oracle.p2p(pos, mass, boxsize=1.0, r_s=r_s, r_cut=r_cut, eps=eps)
    assert np.all(acc == 0.0) and cnt["pairs_in_cut"] == 0
    pos[1] = pos[0] + [0.99 * r_cut, 0, 0]
    a_in, c_in = oracle.p2p(pos, mass, boxsize=1.0, r_s=r_s, r_cut=r_cut, eps=0.1 * r_cut)
    a_out, c_out = oracle.p2p(pos, mass, boxsize=1.0, r_s=r_s, r_cut=r_cut, eps=0.2 * r_cut)
    assert c_in["pairs_in_cut"] == 2 and c_out["pairs_in_cut"] == 0 and np.all(a_out == 0.0)


def test_softened_third_law_and_brute_force(oracle):
    rng = np.random.default_rng(321)
    n, n_pm = 48, 16
    r_s = 1.2 / n_pm
    r_cut = 6 * r_s
    eps = 0.03
    pos = np.mod(rng.random((n, 3)) * 0.5 + 0.8, 1.0)      # straddles the seam
    mass = rng.uniform(0.5, 1.5, n)
    acc, _ = oracle.p2p(pos, mass, boxsize=1.0, r_s=r_s, r_cut=r_cut, eps=eps)
    tot = (mass[:, None] * acc).sum(axis=0)
    assert np.abs(tot).max() <= 1e-12 * (mass[:, None] * np.abs(acc)).sum()
    with mpmath.workdps(30):
        ref = np.zeros((n, 3))
        for i in range(n):
            a = [mpmath.mpf(0)] * 3
            for j in range(n):
                d = [mpmath.mpf(pos[j, k]) - mpmath.mpf(pos[i, k]) for k in range(3)]
                d = [dk - mpmath.nint(dk) for dk in d]
                r2 = sum(dk * dk for dk in d)
                r2e = r2 + mpmath.mpf(eps) ** 2
                if r2 > 0 and r2e < mpmath.mpf(r_cut) ** 2:
                    re = mpmath.sqrt(r2e)
                    x = re / (2 * mpmath.mpf(r_s))
                    T = mpmath.erfc(x) + 2 * x / mpmath.sqrt(mpmath.pi) * mpmath.exp(-x * x)
                    w = mpmath.mpf(mass[j]) * T / re ** 3
                    a = [a[k] + w * d[k] for k in range(3)]
            ref[i] = [float(v) for v in a]
    assert np.abs(acc - ref).max() <= 1e-14 * np.abs(ref).max()
