"""Unit systems of PAPER.md:275 -- oracle.  TEST INFRASTRUCTURE, NOT THE PRODUCT.

The method is defined in normalised quantities (p/(m_e c), E/E_s, cB/E_s); a caller whose arrays are in
another unit system converts, computes, and converts momenta back.  This module holds that definition: the four
multipliers (p, E, B, t) of each system, written out from CODATA 2018 independently of the CUDA side, and the
conversion of arrays (plain numpy multiplications, one rounding each).

  LIBRARY      p/(m_e c), E/E_s, cB/E_s, seconds
  SI           kg m/s, V/m, T, s
  NORM_OMEGA   c = q_e = m_e = 1, reference angular frequency omega [1/s]: E unit m_e c omega/q_e, B unit m_e omega/q_e,
               time unit 1/omega
  NORM_LAMBDA  the same with a reference length lambda [m]: omega = c/lambda
  HL_MEV       Heaviside-Lorentz natural units (hbar = c = 1), energies in MeV: p [MeV], E, B [MeV^2], t [1/MeV];
               q_e = sqrt(4 pi alpha), so E_s = m_e^2/sqrt(4 pi alpha) (the paper's internal system)
"""
import math

import numpy as np

LIBRARY, SI, NORM_OMEGA, NORM_LAMBDA, HL_MEV = 0, 1, 2, 3, 4

C = 299792458.0            # m/s (exact)
H = 6.62607015e-34         # J s (exact)
QE = 1.602176634e-19       # C (exact)
ME = 9.1093837015e-31      # kg
ALPHA = 7.2973525693e-3


def schwinger_field_si():
    """E_s = m_e^2 c^3/(q_e hbar) [V/m] (about 1.32e18 V/m)"""
    hbar = H / (2 * math.pi)
    return ME * ME * C ** 3 / (QE * hbar)


def scales(system, reference=0.0):
    """(p, E, B, t): caller's value times the multiplier = library value"""
    es = schwinger_field_si()
    if system == LIBRARY:
        return 1.0, 1.0, 1.0, 1.0
    if system == SI:
        return 1.0 / (ME * C), 1.0 / es, C / es, 1.0
    if system == NORM_OMEGA:
        f = ME * C * reference / QE / es
        return 1.0, f, f, 1.0 / reference
    if system == NORM_LAMBDA:
        f = ME * C * C / (QE * reference) / es
        return 1.0, f, f, reference / C
    if system == HL_MEV:
        mev = 1e6 * QE
        m = ME * C * C / mev
        f = math.sqrt(4 * math.pi * ALPHA) / (m * m)
        return 1.0 / m, f, f, (H / (2 * math.pi)) / mev
    raise ValueError("unknown unit system")


def to_library(system, reference, p, e, b):
    sp, se, sb, _ = scales(system, reference)
    return ([np.asarray(a, dtype=np.float64) * sp for a in p], [np.asarray(a, dtype=np.float64) * se for a in e],
            [np.asarray(a, dtype=np.float64) * sb for a in b])


def momenta_from_library(system, reference, p):
    sp = scales(system, reference)[0]
    return [np.asarray(a, dtype=np.float64) * (1.0 / sp) for a in p]
