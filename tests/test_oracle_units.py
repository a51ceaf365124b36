"""Pins of the oracle's unit conversions (oracle/units.py) against published constants and against
relations between the systems that hold whatever the constants are."""
import math

import numpy as np

from oracle import units as U


def test_schwinger_field_and_si_scales_match_published_values(orc):
    # E_s = 1.3232855e18 V/m, B_s = E_s/c = 4.4140052e9 T, m_e c = 2.7309245e-22 kg m/s (CODATA-derived, textbooks);
    # PAPER.md:65 quotes E_s ~ 1.32e18 V/m
    assert abs(U.schwinger_field_si() / 1.3232855e18 - 1) < 1e-7
    assert abs(U.schwinger_field_si() / orc.schwinger_field() - 1) < 1e-12      # the C++ oracle's own constant
    sp, se, sb, st = U.scales(U.SI)
    assert abs(1 / sp / 2.7309245e-22 - 1) < 1e-7 and abs(1 / sb / 4.4140052e9 - 1) < 1e-7 and st == 1.0
    assert abs(se * 1.3232855e18 - 1) < 1e-7


def test_heaviside_lorentz_scales():
    sp, se, sb, st = U.scales(U.HL_MEV)
    assert abs(1 / sp / 0.51099895 - 1) < 1e-8                       # m_e c^2 = 0.51099895 MeV
    assert abs(st / 6.582119569e-22 - 1) < 1e-9                      # hbar = 6.582119569e-22 MeV s
    assert abs(1 / se / (0.51099895 ** 2 / math.sqrt(4 * math.pi / 137.035999084)) - 1) < 1e-8   # E_s = m^2/e_HL
    assert se == sb
    # the same field through SI: E_HL [MeV^2] = E_SI * sqrt(eps0) (hbar c)^(3/2) / MeV^2, eps0 = q_e^2/(4 pi alpha hbar c):
    hbar = U.H / (2 * math.pi)
    eps0 = U.QE ** 2 / (4 * math.pi * U.ALPHA * hbar * U.C)
    e_si = 3.7e15
    e_hl = e_si * math.sqrt(eps0) * (hbar * U.C) ** 1.5 / (1e6 * U.QE) ** 2
    assert abs(e_hl * se / (e_si * U.scales(U.SI)[1]) - 1) < 1e-12


def test_normalised_systems_agree_with_si():
    lam = 0.8e-6
    omega = 2 * math.pi * U.C / lam
    so = U.scales(U.NORM_OMEGA, omega)
    sl = U.scales(U.NORM_LAMBDA, U.C / omega)                         # lambda_ref = c/omega
    assert np.allclose(so, sl, rtol=1e-15)
    # a0 = 1 is E = m_e c omega/q_e: 4.0e12 V/m at 0.8 um (textbook: a0 = 0.85 sqrt(I[1e18 W/cm^2]) lambda[um])
    e_si = U.ME * U.C * omega / U.QE
    assert abs(e_si / 4.0138e12 - 1) < 1e-3
    assert abs(so[1] / (e_si * U.scales(U.SI)[1]) - 1) < 1e-14
    assert abs(so[3] * omega - 1) < 1e-15 and so[0] == 1.0


def test_chi_is_unit_independent(orc):
    """the same physical particle described in every system has the same chi ("tables are adimensional")"""
    rng = np.random.default_rng(3)
    n = 1000
    p = [rng.standard_normal(n) * 300 for _ in range(3)]
    e = [rng.standard_normal(n) * 1e-3 for _ in range(3)]
    b = [rng.standard_normal(n) * 1e-3 for _ in range(3)]
    ref = orc.chi(orc.LEPTON, p, e, b)
    for system, r in ((U.SI, 0.0), (U.NORM_OMEGA, 2.35e15), (U.NORM_LAMBDA, 1e-6), (U.HL_MEV, 0.0)):
        sp, se, sb, _ = U.scales(system, r)
        pu, eu, bu = [a / sp for a in p], [a / se for a in e], [a / sb for a in b]
        back = U.to_library(system, r, pu, eu, bu)
        assert np.allclose(orc.chi(orc.LEPTON, *back), ref, rtol=1e-12)
        assert np.allclose(U.momenta_from_library(system, r, back[0])[0], pu[0], rtol=1e-15)
