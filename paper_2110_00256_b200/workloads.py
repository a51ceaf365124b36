"""Seeded synthetic input generators (numpy, host side) -- shared by tests, bench and smoke.

This module holds NONE of the method's arithmetic: it only draws momenta, fields and table
geometries with the shapes and value distributions of BASELINE.json's five configurations
(recipes in DESIGN.md "Inputs").  The same bytes are given to the CUDA library and to the
oracle.  The paper uses no dataset; its own benchmark population is synthetic as well
(PAPER.md:301), so these populations stand in for "the paper's laser-plasma workloads" by
shape only.
"""
import math

import numpy as np

LEPTON, PHOTON = 0, 1

# field amplitude A = chi_target / (KAPPA * gamma): for an isotropic momentum and six independent
# N(0,1) field components the transverse force gamma*|e_perp + n x b| has rms 2*gamma*A.
KAPPA = 2.0


def _rng(seed, *stream):
    return np.random.Generator(np.random.Philox(key=[int(seed), hash_stream(stream)]))


def hash_stream(stream):
    h = 0x9E3779B97F4A7C15
    for s in stream:
        h = ((h ^ int(s)) * 0xBF58476D1CE4E5B9) & 0xFFFFFFFFFFFFFFFF
        h ^= h >> 31
    return h


def table_params(config):
    """Table geometry per configuration (dict of picsarqed_table_params fields)."""
    if config == 1:   # the paper's benchmark set
        return dict(qs_chi_min=1e-3, qs_chi_max=1e3, qs_n_chi=256, qs_xi_min=1e-12, qs_n_xi=256,
                    bw_chi_min=2e-2, bw_chi_max=1e3, bw_n_chi=256, bw_n_xi=256)
    if config in (2, 3, 5):
        return dict(qs_chi_min=1e-4, qs_chi_max=1e3, qs_n_chi=1024, qs_xi_min=1e-12, qs_n_xi=1024,
                    bw_chi_min=1e-2, bw_chi_max=1e3, bw_n_chi=1024, bw_n_xi=1024)
    if config == 4:
        return dict(qs_chi_min=1e-4, qs_chi_max=1e3, qs_n_chi=4096, qs_xi_min=1e-12, qs_n_xi=2048,
                    bw_chi_min=1e-4, bw_chi_max=1e3, bw_n_chi=4096, bw_n_xi=2048, qs_n_chi_2d=2048, bw_n_chi_2d=2048)
    raise ValueError(config)


def isotropic_momenta(rng, n, species, g_lo, g_hi, dtype):
    """direction: normalised Gaussian triple; gamma (or gamma_gamma) log-uniform on [g_lo, g_hi].
    Returns ([px,py,pz], gamma)."""
    d = rng.standard_normal((3, n))
    d /= np.sqrt((d * d).sum(axis=0))
    g = np.exp(rng.uniform(math.log(g_lo), math.log(g_hi), n))
    pm = np.sqrt((g - 1.0) * (g + 1.0)) if species == LEPTON else g
    return [np.ascontiguousarray((pm * d[k]).astype(dtype)) for k in range(3)], g


def gaussian_fields(rng, amp, dtype):
    """six field components = amp * N(0,1); returns ([ex,ey,ez], [bx,by,bz])"""
    n = amp.shape[0]
    f = [np.ascontiguousarray((amp * rng.standard_normal(n)).astype(dtype)) for _ in range(6)]
    return f[:3], f[3:]


def config1(seed=1, n=65536, species=LEPTON, dtype=np.float64):
    """C1: gamma log-uniform [10, 1e4], amplitude log-uniform [1e-5, 1e-2] E_s, chi ~ 1e-3..1e2."""
    rng = _rng(seed, 1, species)
    p, g = isotropic_momenta(rng, n, species, 10.0, 1e4, dtype)
    amp = np.exp(rng.uniform(math.log(1e-5), math.log(1e-2), n))
    e, b = gaussian_fields(rng, amp, dtype)
    return p, e, b


def chi_targeted_momenta(seed, config, n, species, g_lo, g_hi, dtype):
    rng = _rng(seed, config, species, 0)
    return isotropic_momenta(rng, n, species, g_lo, g_hi, dtype)


def chi_targeted_fields(seed, config, step, gamma, chi_lo, chi_hi, dtype):
    """C2/C3: fields re-drawn every step from the seed; target chi log-uniform on [chi_lo, chi_hi],
    amplitude = chi_target / (KAPPA * gamma)."""
    rng = _rng(seed, config, 7, step)
    n = gamma.shape[0]
    chi_t = np.exp(rng.uniform(math.log(chi_lo), math.log(chi_hi), n))
    return gaussian_fields(rng, chi_t / (KAPPA * gamma), dtype)


def config2(seed=2, n=1 << 24, dtype=np.float64):
    """C2 leptons: gamma log-uniform [1e2, 1e5].  Returns (p, gamma); fields via config2_fields."""
    return chi_targeted_momenta(seed, 2, n, LEPTON, 1e2, 1e5, dtype)


def config2_fields(seed, step, gamma, dtype=np.float64):
    return chi_targeted_fields(seed, 2, step, gamma, 1e-3, 1e2, dtype)


def config3(seed=3, n=1 << 24, dtype=np.float32):
    """C3 photons: energy log-uniform [1e2, 1e5] m_e c^2."""
    return chi_targeted_momenta(seed, 3, n, PHOTON, 1e2, 1e5, dtype)


def config3_fields(seed, step, gamma, dtype=np.float32):
    return chi_targeted_fields(seed, 3, step, gamma, 1e-2, 1e3, dtype)


def config5(seed=5, n=1 << 20, species=LEPTON, dtype=np.float32):
    """C5: laser-plasma-like.  Target chi: 90 % lognormal (median 1e-2, sigma_ln 1.5) + 10 % power law
    p(chi) ~ chi^-2 on [1e-2, 1e2], clipped to [1e-6, 1e2].  Fields: linearly polarised plane wave
    e = a cos(phi) x, b = a cos(phi) y with a = a0 hbar omega/(m c^2) = 500 * 3.0329e-6 (0.8 um), phi
    uniform, plus N(0, (0.05 a)^2) noise on all six components.  Direction isotropic; gamma =
    chi_target / (a * 0.75) clamped to [2, 1e5] (photons [4, 1e5]) -- 0.75 ~ rms of cos(phi)(1-cos(theta))."""
    rng = _rng(seed, 5, species)
    a = 500.0 * 3.0329e-6
    body = np.exp(math.log(1e-2) + 1.5 * rng.standard_normal(n))
    u = rng.uniform(size=n)
    tail = 1.0 / (1.0 / 1e-2 - u * (1.0 / 1e-2 - 1.0 / 1e2))  # inverse CDF of chi^-2 on [1e-2, 1e2]
    chi_t = np.clip(np.where(rng.uniform(size=n) < 0.1, tail, body), 1e-6, 1e2)
    g = np.clip(chi_t / (a * 0.75), 2.0 if species == LEPTON else 4.0, 1e5)
    d = rng.standard_normal((3, n))
    d /= np.sqrt((d * d).sum(axis=0))
    pm = np.sqrt((g - 1.0) * (g + 1.0)) if species == LEPTON else g
    p = [np.ascontiguousarray((pm * d[k]).astype(dtype)) for k in range(3)]
    wave = a * np.cos(rng.uniform(0.0, 2.0 * math.pi, n))
    f = [0.05 * a * rng.standard_normal(n) for _ in range(6)]
    f[0] += wave
    f[4] += wave
    f = [np.ascontiguousarray(x.astype(dtype)) for x in f]
    return p, f[:3], f[3:]


def choose_dt(rates, target=0.05):
    """dt such that mean(1 - exp(-R dt)) = target over the given rates (1/s), by bisection."""
    r = np.asarray(rates, dtype=np.float64)
    r = r[np.isfinite(r) & (r > 0)]
    lo, hi = 0.0, 1.0 / r.mean()
    while np.mean(-np.expm1(-r * hi)) < target:
        hi *= 2.0
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if np.mean(-np.expm1(-r * mid)) < target:
            lo = mid
        else:
            hi = mid
    return 0.5 * (lo + hi)
