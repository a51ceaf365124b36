"""Pins for the table half of the oracle (oracle/picsarqed_oracle.cpp, part I).

Nothing here compares the oracle with itself or with the CUDA path: every expectation is a
library routine (mpmath / scipy), a closed form, an asymptotic limit, a symmetry, or a value
computed independently during the survey (tests/golden/survey_table_values.txt).
"""
import math

import mpmath as mp
import numpy as np
import pytest
import scipy.special as sps
from scipy.integrate import quad

from conftest import golden

mp.mp.dps = 30
SQ3 = math.sqrt(3.0)


# ----------------------------------------------------------------------------- quadrature rule
def test_gk15_constants_are_exact_for_polynomials(orc):
    assert orc.selftest_gk15() < 5e-16


# ----------------------------------------------------------------------------- Bessel K, IK
@pytest.mark.parametrize("nu", [1 / 3, 2 / 3, 5 / 3, 0.5])
@pytest.mark.parametrize("x", [1e-18, 1e-9, 1e-3, 0.3, 1.0, 7.0, 66.0, 700.0, 4e4])
def test_bessel_k_scaled_vs_mpmath(orc, nu, x):
    ref = float(mp.besselk(nu, x) * mp.exp(x))
    assert orc.bessel_k_scaled(nu, x) == pytest.approx(ref, rel=2e-14)


@pytest.mark.parametrize("x", [0.05, 1.0, 30.0, 300.0])
def test_bessel_k_vs_library_kv_and_half_order_closed_form(orc, x):
    # scipy's kve is the exponentially scaled library routine (AMOS)
    for nu in (1 / 3, 2 / 3):
        assert orc.bessel_k_scaled(nu, x) == pytest.approx(sps.kve(nu, x), rel=1e-13)
    # K_{1/2}(x) = sqrt(pi/2x) e^{-x}
    assert orc.bessel_k_scaled(0.5, x) == pytest.approx(math.sqrt(math.pi / (2 * x)), rel=2e-15)


@pytest.mark.parametrize("x", [0.2, 1.0, 2.5, 6.0])
def test_airy_relations(orc, x):
    # Ai(x) = (1/pi) sqrt(x/3) K_{1/3}(z), Ai'(x) = -(x/(pi sqrt3)) K_{2/3}(z), z = (2/3) x^{3/2}
    z = 2 / 3 * x ** 1.5
    ai, aip, _, _ = sps.airy(x)
    assert math.sqrt(x / 3) / math.pi * orc.bessel_k_scaled(1 / 3, z) * math.exp(-z) == pytest.approx(ai, rel=1e-13)
    assert -x / (math.pi * SQ3) * orc.bessel_k_scaled(2 / 3, z) * math.exp(-z) == pytest.approx(aip, rel=1e-13)


def test_recurrence_k53(orc):
    # K_{5/3}(x) = K_{1/3}(x) + (4/(3x)) K_{2/3}(x)
    for x in (0.01, 1.0, 20.0):
        lhs = orc.bessel_k_scaled(5 / 3, x)
        rhs = orc.bessel_k_scaled(1 / 3, x) + 4 / (3 * x) * orc.bessel_k_scaled(2 / 3, x)
        assert lhs == pytest.approx(rhs, rel=1e-13)


@pytest.mark.parametrize("nu,x", [(1 / 3, 1e-3), (1 / 3, 1.0), (1 / 3, 100.0), (5 / 3, 1e-6), (5 / 3, 2.5),
                                  (2 / 3, 12.0)])
def test_bessel_ik_scaled_vs_quadrature_of_library_k(orc, nu, x):
    # int_x^inf K_nu(t) dt by QUADPACK over the library's (scaled) K_nu
    pts = sorted({x, min(2 * x, x + 0.5), x + 1, x + 10, x + 50})
    ref = sum(quad(lambda t: sps.kve(nu, t) * math.exp(x - t), a, b, epsabs=0, epsrel=1e-13, limit=200)[0]
              for a, b in zip(pts[:-1], pts[1:]) if b > a)
    assert orc.bessel_ik_scaled(nu, x) == pytest.approx(ref, rel=2e-12)


def test_bessel_ik_scaled_vs_mpmath(orc):
    nu, x = 1 / 3, 1.0
    ref = float(mp.quad(lambda t: mp.besselk(nu, t) * mp.exp(x), mp.linspace(x, x + 40, 21) + [mp.inf]))
    assert orc.bessel_ik_scaled(nu, x) == pytest.approx(ref, rel=1e-14)


def test_ik13_at_zero_closed_form(orc):
    # int_0^inf K_{1/3} = pi / (2 cos(pi/6)) = pi/sqrt(3); int_0^x K_{1/3} ~ small for x = 1e-15
    x = 1e-15
    head = float(mp.quad(lambda t: mp.besselk(1 / 3, t), [0, x]))
    assert orc.bessel_ik_scaled(1 / 3, x) * math.exp(-x) == pytest.approx(math.pi / SQ3 - head, rel=1e-14)


# ----------------------------------------------------------------------------- integrands, literal forms
@pytest.mark.parametrize("chi,xi", [(0.3, 0.4), (1.0, 0.25), (3.0, 0.07), (30.0, 0.5), (1000.0, 0.9)])
def test_bw_integrand_vs_literal_eq4(orc, chi, xi):
    """eq.4/eq.9 bracket evaluated literally with mpmath: X = (chi_g/(chi_+ chi_-))^{2/3},
    int_X^inf sqrt(s) K_{1/3}((2/3)s^{3/2}) ds - (2 - chi_g X^{3/2}) K_{2/3}((2/3) X^{3/2})"""
    chim, chip = xi * chi, (1 - xi) * chi
    X = (mp.mpf(chi) / (chim * chip)) ** (mp.mpf(2) / 3)
    inner = mp.quad(lambda s: mp.sqrt(s) * mp.besselk(mp.mpf(1) / 3, mp.mpf(2) / 3 * s ** 1.5),
                    [X, X + 1, X + 5, X + 30, mp.inf])
    lit = inner - (2 - chi * X ** 1.5) * mp.besselk(mp.mpf(2) / 3, mp.mpf(2) / 3 * X ** 1.5)
    got = mp.mpf(orc.bw_f_scaled(chi, xi)) * mp.exp(-mp.mpf(8) / (3 * chi))
    assert float(got / lit) == pytest.approx(1.0, abs=1e-12)


@pytest.mark.parametrize("chi,xi", [(0.01, 1e-3), (0.3, 0.2), (1.0, 1e-9), (1.0, 0.5), (30.0, 0.95), (1e3, 0.999)])
def test_qs_integrand_vs_literal_eq12(orc, chi, xi):
    """S/xi = sqrt3/(2 pi) [ int_Y^inf K_{5/3} + xi^2/(1-xi) K_{2/3}(Y) ], Y = 2xi/(3chi(1-xi))"""
    Y = mp.mpf(2) * xi / (3 * mp.mpf(chi) * (1 - mp.mpf(xi)))
    ik = mp.quad(lambda s: mp.besselk(mp.mpf(5) / 3, s), [Y, 2 * Y, 10 * Y + 1, 10 * Y + 40, mp.inf])
    lit = mp.sqrt(3) / (2 * mp.pi) * (ik + mp.mpf(xi) ** 2 / (1 - mp.mpf(xi)) * mp.besselk(mp.mpf(2) / 3, Y))
    assert orc.qs_s_over_xi(chi, xi) == pytest.approx(float(lit), rel=1e-12)


def test_bw_T_literal_nested_eq9(orc):
    """T from the literal double integral of eq.9, QUADPACK over the library K_nu"""
    for chi in (1.0, 10.0):
        def bracket(u):
            X = (chi / (u * (chi - u))) ** (2 / 3)
            inner = quad(lambda s: math.sqrt(s) * sps.kv(1 / 3, 2 / 3 * s ** 1.5), X, np.inf, epsabs=0, epsrel=1e-12)[0]
            return inner - (2 - chi * X ** 1.5) * sps.kv(2 / 3, 2 / 3 * X ** 1.5)
        T = quad(bracket, 0, chi, epsabs=0, epsrel=1e-11, limit=200)[0] / (math.pi * SQ3 * chi ** 2)
        assert math.exp(orc.bw_lnT(chi)) == pytest.approx(T, rel=1e-9)


# ----------------------------------------------------------------------------- T and G: values and limits
def test_T_G_survey_values(orc):
    for kind, chi, _, val in golden("survey_table_values.txt"):
        chi, val = float(chi), float(val)
        if kind == "T":
            assert math.exp(orc.bw_lnT(chi)) == pytest.approx(val, rel=2e-9)
        elif kind == "lnT":
            assert orc.bw_lnT(chi) == pytest.approx(val, abs=2e-7)
        elif kind == "G":
            assert orc.qs_G(chi) == pytest.approx(val, rel=2e-9)


def test_T_small_chi_limit(orc):
    # T e^{8/(3 chi)} -> 3 sqrt3 / (16 sqrt2) (saddle point of eq.9), corrections O(chi)
    lim = 3 * SQ3 / (16 * math.sqrt(2))
    d3 = orc.bw_T_scaled(1e-3) / lim - 1
    d4 = orc.bw_T_scaled(1e-4) / lim - 1
    assert abs(d4) < 3e-5 and abs(d3) < 3e-4
    assert d3 / d4 == pytest.approx(10.0, rel=0.05)  # first-order in chi
    # the paper's statement T ~ exp(-8/(3 chi)) for chi << 1 (eq.10 with the corrected argument)
    assert orc.bw_lnT(1e-3) == pytest.approx(-8 / 3e-3 + math.log(lim), abs=1e-3)


def test_T_large_chi_limit(orc):
    # T chi^{1/3} -> (1/(pi sqrt3)) (Gamma(2/3)/2) 3^{2/3} [B(2/3,2/3) - 2 B(5/3,5/3)]
    g = math.gamma
    B = lambda a, b: g(a) * g(b) / g(a + b)
    lim = (1 / (math.pi * SQ3)) * (g(2 / 3) / 2) * 3 ** (2 / 3) * (B(2 / 3, 2 / 3) - 2 * B(5 / 3, 5 / 3))
    assert lim == pytest.approx(0.3796123085, rel=1e-9)
    dev = [math.exp(orc.bw_lnT(c)) * c ** (1 / 3) / lim - 1 for c in (1e4, 1e6, 1e8)]
    assert abs(dev[0]) < 1e-2 and abs(dev[1]) < abs(dev[0]) / 5 and abs(dev[2]) < abs(dev[1]) / 5


def test_G_limits(orc):
    # chi -> 0: classical photon emission rate, G/chi -> 5 sqrt3/4 ; chi -> inf: G/chi^{2/3} -> const
    lo = 5 * SQ3 / 4
    d = [orc.qs_G(c) / c / lo - 1 for c in (1e-3, 1e-4, 1e-5)]
    assert abs(d[2]) < 2e-5 and d[0] / d[1] == pytest.approx(10, rel=0.05)
    g = math.gamma
    B = lambda a, b: g(a) * g(b) / g(a + b)
    hi = (SQ3 / (2 * math.pi)) * g(2 / 3) * 3 ** (2 / 3) * (B(1 / 3, 5 / 3) + 0.5 * B(7 / 3, 2 / 3))
    assert hi == pytest.approx(2.1907501936, rel=1e-9)
    dev = [orc.qs_G(c) / c ** (2 / 3) / hi - 1 for c in (1e3, 1e4, 1e5)]
    assert abs(dev[0]) < 0.15 and abs(dev[1]) < abs(dev[0]) / 1.5 and abs(dev[2]) < abs(dev[1]) / 1.5


def test_qs_first_moment_classical_power(orc):
    # int_0^1 S dxi -> chi^2 (classical radiated power) as chi -> 0
    d = [orc.qs_first_moment(c) / c ** 2 - 1 for c in (1e-3, 1e-4)]
    assert abs(d[1]) < 1e-3 and d[0] / d[1] == pytest.approx(10, rel=0.1)


def test_erber_form_is_the_corrected_one(orc):
    """PAPER.md:203 uses eq.10 outside the T table; with the argument 4/(3 chi) (R2) it is a
    0.82..0.99 approximation of eq.9; with the printed 2/(3 chi) it would be off by 1.6x..1e6x."""
    for chi, lo, hi in ((0.05, 0.80, 0.84), (1.0, 0.84, 0.87), (10.0, 0.91, 0.93), (1000.0, 0.98, 0.99)):
        ratio = orc.erber_T(chi) / math.exp(orc.bw_lnT(chi))
        assert lo < ratio < hi
    # value of the form itself, from the library Bessel function
    assert orc.erber_T(2.0) == pytest.approx(0.16 * sps.kv(1 / 3, 4 / 6.0) ** 2 / 2.0, rel=1e-13)
    assert orc.erber_T(0.0) == 0.0


# ----------------------------------------------------------------------------- CDFs
def test_cdf_survey_values(orc):
    for kind, chi, xi, val in golden("survey_table_values.txt"):
        if kind == "PBW":
            assert orc.bw_cdf(float(chi), float(xi)) == pytest.approx(float(val), rel=3e-9, abs=6e-11)
        elif kind == "PQS":
            assert orc.qs_cdf(float(chi), float(xi)) == pytest.approx(float(val), rel=3e-9, abs=6e-11)


def test_bw_cdf_symmetry(orc):
    # P(chi, xi) = 1 - P(chi, 1 - xi)
    for chi in (0.1, 1.0, 50.0):
        assert orc.bw_cdf(chi, 0.5) == pytest.approx(0.5, abs=1e-12)
        for xi in (0.2, 0.35):
            assert orc.bw_cdf(chi, xi) + orc.bw_cdf(chi, 1 - xi) == pytest.approx(1.0, abs=1e-12)


def test_qs_cdf_small_xi_power_law(orc):
    # P ~ c xi^{1/3},  c = (sqrt3/2pi) 2^{2/3} Gamma(2/3) (3 chi/2)^{2/3} 3 / G(chi)
    for chi in (1e-2, 1.0, 100.0):
        c = SQ3 / (2 * math.pi) * 2 ** (2 / 3) * math.gamma(2 / 3) * (1.5 * chi) ** (2 / 3) * 3 / orc.qs_G(chi)
        assert orc.qs_cdf(chi, 1e-12) == pytest.approx(c * 1e-4, rel=2e-3)


def test_table_rows(orc, small_tables):
    t, p = small_tables, small_tables.params
    # BW rows: P(1/2) computed = 1/2 before being fixed; non-decreasing; first 0, last 0.5
    rows, half = orc.build_bw_rows(p, 3, 6, return_half=True)
    assert np.allclose(half, 0.5, atol=1e-12)
    assert np.all(np.diff(t.bw_P, axis=1) >= 0) and np.all(t.bw_P[:, 0] == 0) and np.all(t.bw_P[:, -1] == 0.5)
    # QS rows: row total = G(chi_n); ln P non-decreasing, last exactly 0
    rows, tot = orc.build_qs_rows(p, 0, p.qs_n_chi, return_total=True)
    assert np.allclose(np.log(tot), t.lnG, atol=1e-11)
    assert np.all(np.diff(t.qs_lnP, axis=1) >= 0) and np.all(t.qs_lnP[:, -1] == 0)
    # entries are the CDF definitions at the grid points
    chis = np.exp(np.linspace(math.log(p.bw_chi_min), math.log(p.bw_chi_max), p.bw_n_chi))
    for n, m in ((5, 30), (12, 17), (24, 40)):
        assert t.bw_P[n, m] == pytest.approx(orc.bw_cdf(chis[n], 0.5 * m / (p.bw_n_xi - 1)), rel=1e-10, abs=1e-300)
    chis = np.exp(np.linspace(math.log(p.qs_chi_min), math.log(p.qs_chi_max), p.qs_n_chi))
    for n, m in ((0, 0), (7, 20), (24, 47)):
        xi = p.qs_xi_min ** (1 - m / (p.qs_n_xi - 1))
        assert t.qs_lnP[n, m] == pytest.approx(math.log(orc.qs_cdf(chis[n], xi)), abs=1e-10)
    # 1D tables at their nodes
    assert t.lnT[10] == pytest.approx(orc.bw_lnT(math.exp(math.log(p.bw_chi_min) + 10 * math.log(p.bw_chi_max / p.bw_chi_min) / (p.bw_n_chi - 1))), abs=1e-12)
    assert t.lnG[0] == pytest.approx(math.log(orc.qs_G(p.qs_chi_min)), abs=1e-13)


def test_small_chi_gamma_rows_do_not_underflow(orc):
    # chi_gamma = 1e-4: ln T ~ -26668, yet the CDF row is a proper CDF (scaled evaluation, R9)
    p = orc.TableParams(bw_chi_min=1e-4, bw_chi_max=1e-3, bw_n_chi=2, bw_n_xi=33)
    rows = orc.build_bw_rows(p, 0, 1)
    assert rows[0, -1] == 0.5 and rows[0, -2] > 0 and np.all(np.diff(rows[0]) >= 0)
    sigma = math.sqrt(3 * 1e-4 / 64)  # Gaussian bump of that width around 1/2
    xi = 0.5 - 0.5 / 32
    assert rows[0, -2] == pytest.approx(0.5 * math.erfc((0.5 - xi) / (sigma * math.sqrt(2))), rel=0.05)
