"""Pins for the runtime half of the oracle (oracle/picsarqed_oracle.cpp, part II).

Expectations are the paper's worked values (tests/golden), closed forms, invariances,
conservation laws, published known-answer vectors and brute-force Monte Carlo frequencies.
"""
import math

import numpy as np
import pytest
import scipy.stats as st

from conftest import golden

LEPTON, PHOTON, F32, F64 = 0, 1, 0, 1
ALPHA_OVER_TAUC = 7.2973525693e-3 * 9.1093837015e-31 * 299792458.0 ** 2 / (6.62607015e-34 / (2 * math.pi))


def vec(*rows):
    """rows of (x,y,z) -> three arrays"""
    a = np.array(rows, dtype=np.float64).reshape(-1, 3)
    return a[:, 0].copy(), a[:, 1].copy(), a[:, 2].copy()


# ----------------------------------------------------------------------------- constants
def test_schwinger_field_and_prefactor(orc):
    assert orc.schwinger_field() == pytest.approx(1.32e18, rel=3e-3)
    assert orc.schwinger_field() == pytest.approx(1.3232854741e18, rel=1e-9)  # CODATA 2018
    assert orc.rate_prefactor() == pytest.approx(ALPHA_OVER_TAUC, rel=1e-14)
    assert orc.rate_prefactor() == pytest.approx(5.6652563985e18, rel=1e-9)


# ----------------------------------------------------------------------------- chi
def test_chi_paper_worked_cases(orc):
    for name, g0, kind, amp, expect, tol in golden("paper_chi_cases.txt"):
        g0, amp, expect, tol = float(g0), float(amp), float(expect), float(tol)
        pmag = math.sqrt(g0 * g0 - 1)
        if kind == "perp_B":      # p along x, B along z
            p, e, b = vec((pmag, 0, 0)), vec((0, 0, 0)), vec((0, 0, amp))
        else:                     # wave travelling along -x: E along y, B = k_hat x E = -x_hat x y_hat E = -z E
            p, e, b = vec((pmag, 0, 0)), vec((0, amp, 0)), vec((0, 0, -amp))
        assert orc.chi(LEPTON, p, e, b)[0] == pytest.approx(expect, rel=tol), name


def test_chi_closed_forms(orc):
    # p perpendicular to b only: chi = |p| |b| (both species)
    p, e, b = vec((300.0, 0, 0)), vec((0, 0, 0)), vec((0, 2e-3, 0))
    assert orc.chi(LEPTON, p, e, b)[0] == pytest.approx(0.6, rel=1e-15)
    assert orc.chi(PHOTON, p, e, b)[0] == pytest.approx(0.6, rel=1e-15)
    # e parallel to p only: lepton chi = |e| (gamma^2 - p^2 = 1), photon chi = 0
    p, e, b = vec((300.0, 0, 0)), vec((2e-3, 0, 0)), vec((0, 0, 0))
    assert orc.chi(LEPTON, p, e, b)[0] == pytest.approx(2e-3, rel=1e-15)
    assert orc.chi(PHOTON, p, e, b)[0] == 0.0
    # head-on plane wave: chi = (gamma + |p|) E0 ; co-propagating: (gamma - |p|) E0
    pm = 4000.0
    g = math.sqrt(1 + pm * pm)
    p, e = vec((pm, 0, 0)), vec((0, 1e-4, 0))
    assert orc.chi(LEPTON, p, e, vec((0, 0, -1e-4)))[0] == pytest.approx((g + pm) * 1e-4, rel=1e-15)
    assert orc.chi(LEPTON, p, e, vec((0, 0, 1e-4)))[0] == pytest.approx(1e-4 / (g + pm), rel=1e-12)
    assert orc.chi(PHOTON, p, e, vec((0, 0, 1e-4)))[0] == pytest.approx(0.0, abs=1e-20)


def _boost(p4, E, B, beta):
    """Lorentz boost with velocity beta (3-vector, units of c) of a 4-momentum and of (E, cB)."""
    beta = np.asarray(beta, float)
    b2 = beta @ beta
    g = 1 / math.sqrt(1 - b2)
    n = beta / math.sqrt(b2)
    en, pv = p4[0], p4[1:]
    ppar = pv @ n
    en2 = g * (en - math.sqrt(b2) * ppar)
    pv2 = pv + ((g - 1) * ppar - g * math.sqrt(b2) * en) * n
    E2 = g * (E + np.cross(beta, B)) - (g - 1) * (E @ n) * n
    B2 = g * (B - np.cross(beta, E)) - (g - 1) * (B @ n) * n
    return np.concatenate([[en2], pv2]), E2, B2


def test_chi_is_lorentz_invariant_and_homogeneous(orc):
    rng = np.random.default_rng(5)
    for species in (LEPTON, PHOTON):
        for _ in range(20):
            pv = rng.normal(size=3) * 50
            E, B = rng.normal(size=3) * 1e-3, rng.normal(size=3) * 1e-3
            en = math.sqrt((1 if species == LEPTON else 0) + pv @ pv)
            c0 = orc.chi(species, vec(pv), vec(E), vec(B))[0]
            p4, E2, B2 = _boost(np.concatenate([[en], pv]), E, B, rng.normal(size=3) * 0.3)
            c1 = orc.chi(species, vec(p4[1:]), vec(E2), vec(B2))[0]
            assert c1 == pytest.approx(c0, rel=1e-10)
            c2 = orc.chi(species, vec(pv), vec(3.5 * E), vec(3.5 * B))[0]
            assert c2 == pytest.approx(3.5 * c0, rel=1e-14)


# ----------------------------------------------------------------------------- Philox and uniforms
def test_philox_known_answers(orc):
    for row in golden("philox4x32_10_kat.txt"):
        w = [int(x, 16) for x in row]
        assert orc.philox4x32_10(w[0:4], w[4:6]) == tuple(w[6:10])


def test_uniforms_open_interval_and_distribution(orc):
    for dtype, tiny in ((F64, 2.0 ** -53), (F32, 2.0 ** -24)):
        u = np.array([orc.uniform(7, i, 3, 1, 0, i % 2, dtype) for i in range(20000)])
        assert u.min() >= tiny and u.max() <= 1 - tiny
        assert st.kstest(u, "uniform").pvalue > 1e-3
        if dtype == F32:
            assert np.all(u == u.astype(np.float32))  # exactly representable in the target type
    # streams differ by every counter field
    base = orc.uniform(1, 2, 3, 1, 0, 0, F64)
    others = [orc.uniform(2, 2, 3, 1, 0, 0, F64), orc.uniform(1, 3, 3, 1, 0, 0, F64),
              orc.uniform(1, 2, 4, 1, 0, 0, F64), orc.uniform(1, 2, 3, 2, 0, 0, F64),
              orc.uniform(1, 2, 3, 1, 1, 0, F64), orc.uniform(1, 2, 3, 1, 0, 1, F64),
              orc.uniform(1, 2 + 2 ** 32, 3, 1, 0, 0, F64), orc.uniform(1, 2, 3 + 2 ** 32, 1, 0, 0, F64)]
    assert len({base, *others}) == 9


def test_initial_optical_depth_is_exponential(orc):
    for tdt in (F64, F32):
        tau = orc.init_optical_depth(LEPTON, tdt, 200000, seed=11)
        assert np.all(np.isfinite(tau)) and tau.min() > 0
        assert tau.mean() == pytest.approx(1.0, abs=4 / math.sqrt(2e5))
        assert tau.var() == pytest.approx(1.0, abs=0.03)
        assert st.kstest(tau, "expon").pvalue > 1e-3
    # tau = -ln U with the documented stream (purpose 0, step 0, words 0,1)
    t0 = orc.init_optical_depth(PHOTON, F64, 3, seed=5, ids=np.array([9, 10, 2 ** 40], dtype=np.uint64))
    for t, i in zip(t0, (9, 10, 2 ** 40)):
        assert t == pytest.approx(-math.log(orc.uniform(5, i, 0, 0, PHOTON, 0, F64)), rel=1e-15)


# ----------------------------------------------------------------------------- 1D lookups and rates
def _power_law_tables(orc, read_fp32=False):
    """tables whose entries are exact power laws, so eqs.23/27 must reproduce them exactly"""
    p = orc.TableParams(qs_chi_min=1e-3, qs_chi_max=1e2, qs_n_chi=17, qs_xi_min=1e-6, qs_n_xi=9,
                        bw_chi_min=1e-1, bw_chi_max=1e2, bw_n_chi=13, bw_n_xi=9)
    lq = np.linspace(math.log(p.qs_chi_min), math.log(p.qs_chi_max), p.qs_n_chi)
    lb = np.linspace(math.log(p.bw_chi_min), math.log(p.bw_chi_max), p.bw_n_chi)
    lnG = 0.3 + 0.8 * lq
    lnT = -1.0 - 0.4 * lb
    # CDF rows independent of chi: QS P = xi^{1/3} -> ln P = ln(xi)/3 ; BW P = xi (uniform split)
    lxi = math.log(p.qs_xi_min) * (1 - np.arange(p.qs_n_xi) / (p.qs_n_xi - 1))
    qs = np.tile(lxi / 3, (p.qs_n_chi, 1))
    bw = np.tile(0.5 * np.arange(p.bw_n_xi) / (p.bw_n_xi - 1), (p.bw_n_chi, 1))
    return orc.Tables(p, lnG, qs, lnT, bw, read_fp32)


def test_rate_power_law_tables_and_clamps(orc):
    t = _power_law_tables(orc)
    # lepton, p perp b: chi = |p||b|
    for chi_want in (1e-3, 0.02, 0.7, 55.0, 1e2):
        pm = 1000.0
        g = math.sqrt(1 + pm * pm)
        r = orc.rate(t, LEPTON, vec((pm, 0, 0)), vec((0, 0, 0)), vec((0, chi_want / pm, 0)))[0]
        G = math.exp(0.3) * chi_want ** 0.8
        assert r == pytest.approx(2 / 3 * ALPHA_OVER_TAUC * G / g, rel=1e-13)   # eq.15 + eq.27
    # outside the G table: first / last value
    for chi_want, edge in ((1e-5, 1e-3), (5e3, 1e2), (0.0, 1e-3)):
        pm = 1000.0
        r = orc.rate(t, LEPTON, vec((pm, 0, 0)), vec((0, 0, 0)), vec((0, chi_want / pm, 0)))[0]
        assert r == pytest.approx(2 / 3 * ALPHA_OVER_TAUC * math.exp(0.3) * edge ** 0.8 / math.sqrt(1 + pm * pm), rel=1e-13)
    # photon inside the T table: eq.8 + eq.23
    for chi_want in (0.11, 3.0, 90.0):
        pm = 500.0
        r = orc.rate(t, PHOTON, vec((0, pm, 0)), vec((0, 0, 0)), vec((chi_want / pm, 0, 0)))[0]
        assert r == pytest.approx(ALPHA_OVER_TAUC * chi_want * math.exp(-1.0) * chi_want ** -0.4 / pm, rel=1e-13)
    # outside: Erber form; photons that cannot make a pair: 0
    for chi_want in (0.05, 400.0):
        pm = 500.0
        r = orc.rate(t, PHOTON, vec((0, pm, 0)), vec((0, 0, 0)), vec((chi_want / pm, 0, 0)))[0]
        assert r == pytest.approx(ALPHA_OVER_TAUC * chi_want * orc.erber_T(chi_want) / pm, rel=1e-12)
    assert orc.rate(t, PHOTON, vec((0, 1.9, 0)), vec((0, 0, 0)), vec((1.0, 0, 0)))[0] == 0.0
    assert orc.rate(t, PHOTON, vec((0, 0, 0)), vec((0, 0, 0)), vec((1.0, 0, 0)))[0] == 0.0


def test_rate_fp32_table_reads(orc):
    t64, t32 = _power_law_tables(orc), _power_law_tables(orc, read_fp32=True)
    a = (vec((1000.0, 0, 0)), vec((0, 0, 0)), vec((0, 3e-4, 0)))
    r64, r32 = orc.rate(t64, LEPTON, *a)[0], orc.rate(t32, LEPTON, *a)[0]
    assert r32 != r64 and r32 == pytest.approx(r64, rel=1e-6)


def test_classical_synchrotron_photon_rate(orc, small_tables):
    # textbook: dN/dt = (5/(2 sqrt3)) alpha (e B/m) for chi << 1, i.e. (5/(2 sqrt3)) (alpha/tau_C) b
    b = 2e-6
    r = orc.rate(small_tables, LEPTON, vec((1000.0, 0, 0)), vec((0, 0, 0)), vec((0, 0, b)))[0]
    assert r == pytest.approx(5 / (2 * math.sqrt(3)) * ALPHA_OVER_TAUC * b, rel=5e-3)


def test_pair_rate_small_chi_textbook(orc):
    # W = (3 sqrt3/(16 sqrt2)) (alpha/tau_C) (chi/gamma_g) e^{-8/(3chi)} for chi << 1; build a T table around it
    p = orc.TableParams(bw_chi_min=0.05, bw_chi_max=0.2, bw_n_chi=33, bw_n_xi=3, qs_n_chi=2, qs_n_xi=2)
    t = orc.Tables(p, np.zeros(2), np.zeros((2, 2)), orc.build_lnT(p), np.tile([0, .25, .5], (33, 1)))
    chi, pm = 0.1, 400.0
    r = orc.rate(t, PHOTON, vec((pm, 0, 0)), vec((0, 0, 0)), vec((0, chi / pm, 0)))[0]
    W = 3 * math.sqrt(3) / (16 * math.sqrt(2)) * ALPHA_OVER_TAUC * chi / pm * math.exp(-8 / (3 * chi))
    assert r == pytest.approx(W, rel=0.05)   # first correction is O(chi)


# ----------------------------------------------------------------------------- evolve + event frequency
def test_evolve_decrements_by_rate_dt(orc, small_tables):
    rng = np.random.default_rng(2)
    n = 64
    p = [rng.normal(size=n) * 300 for _ in range(3)]
    e = [rng.normal(size=n) * 1e-3 for _ in range(3)]
    b = [rng.normal(size=n) * 1e-3 for _ in range(3)]
    tau = rng.exponential(size=n)
    for sp in (LEPTON, PHOTON):
        R = orc.rate(small_tables, sp, p, e, b)
        o = orc.evolve_optical_depth(small_tables, sp, F64, p, e, b, 1e-17, tau)
        assert np.allclose(o["tau"], tau - R * 1e-17, rtol=0, atol=1e-15)
        assert np.allclose(o["decr"], R * 1e-17, rtol=1e-14)
        o32 = orc.evolve_optical_depth(small_tables, sp, F32, p, e, b, 1e-17, tau)
        assert np.all(o32["tau"] == o["tau_exact"].astype(np.float32))


def test_event_frequency_matches_integrated_rate(orc, small_tables):
    """brute force: fraction with tau < 0 after one step = 1 - exp(-R dt);
    after k steps survival = exp(-k R dt)"""
    n = 400000
    for sp, pm, bfield in ((LEPTON, 1000.0, 1e-3), (PHOTON, 2000.0, 1.5e-3)):
        p = [np.full(n, pm), np.zeros(n), np.zeros(n)]
        e = [np.zeros(n)] * 3
        b = [np.zeros(n), np.zeros(n), np.full(n, bfield)]
        R = orc.rate(small_tables, sp, p, e, b)[0]
        dt = 0.05 / R
        tau = orc.init_optical_depth(sp, F64, n, seed=3)
        alive = np.ones(n, bool)
        for k in (1, 2, 3):
            tau = orc.evolve_optical_depth(small_tables, sp, F64, p, e, b, dt, tau)["tau"]
            frac = np.mean(tau < 0)
            expect = 1 - math.exp(-k * R * dt)
            assert abs(frac - expect) < 4 * math.sqrt(expect * (1 - expect) / n)


# ----------------------------------------------------------------------------- events
def _population(rng, n, species, gmin=10, gmax=1e4):
    d = rng.normal(size=(3, n))
    d /= np.linalg.norm(d, axis=0)
    g = np.exp(rng.uniform(math.log(gmin), math.log(gmax), n))
    pm = np.sqrt(g * g - 1) if species == LEPTON else g
    amp = np.exp(rng.uniform(math.log(1e-5), math.log(1e-2), n))
    e = [amp * rng.normal(size=n) for _ in range(3)]
    b = [amp * rng.normal(size=n) for _ in range(3)]
    return [pm * d[0], pm * d[1], pm * d[2]], e, b, g


def test_photon_emission_conserves_energy_and_direction(orc, small_tables):
    rng = np.random.default_rng(0)
    n = 3000
    p, e, b, g = _population(rng, n, LEPTON)
    tau = np.where(rng.random(n) < 0.4, -rng.random(n), rng.random(n) + 0.1)
    o = orc.generate_photons(small_tables, F64, F64, p, e, b, tau, seed=9, step=4)
    fired = np.flatnonzero(tau < 0)
    assert o["n_fired"] == fired.size and np.array_equal(o["parent"], fired)      # index order
    gph = np.sqrt(sum(c * c for c in o["ph_p"]))
    g_after = np.sqrt(1 + sum(c * c for c in o["p"]))
    assert np.allclose(g_after[fired] + gph, g[fired], rtol=1e-12)
    assert np.allclose(gph, (g[fired] - 1) * o["xi"], rtol=1e-12)
    assert np.all((o["xi"] > 0) & (o["xi"] < 1))
    for k in range(3):  # emitted along p; emitter keeps its direction
        assert np.allclose(o["ph_p"][k] / gph, p[k][fired] / np.sqrt(g[fired] ** 2 - 1), atol=1e-12)
        assert np.allclose(o["p"][k][fired] / np.sqrt(g_after[fired] ** 2 - 1), p[k][fired] / np.sqrt(g[fired] ** 2 - 1), atol=1e-9)
    keep = np.flatnonzero(tau >= 0)
    assert all(np.array_equal(o["p"][k][keep], p[k][keep]) for k in range(3))
    assert np.array_equal(o["tau"][keep], tau[keep])
    assert np.all(o["tau"][fired] > 0) and np.all(o["ph_tau"] > 0)
    # the re-drawn optical depths follow the documented stream
    i = int(fired[5])
    assert o["tau"][i] == pytest.approx(-math.log(orc.uniform(9, i, 4, 1, LEPTON, 1, F64)), rel=1e-15)
    assert o["ph_tau"][5] == pytest.approx(-math.log(orc.uniform(9, i, 4, 2, LEPTON, 0, F64)), rel=1e-15)


def test_pair_production_conserves_energy(orc, small_tables):
    rng = np.random.default_rng(1)
    n = 3000
    p, e, b, g = _population(rng, n, PHOTON)
    tau = np.where(rng.random(n) < 0.4, -rng.random(n), rng.random(n) + 0.1)
    o = orc.generate_pairs(small_tables, F64, F64, p, e, b, tau, seed=9, step=4)
    fired = np.flatnonzero(tau < 0)
    assert o["n_fired"] == fired.size and np.array_equal(o["parent"], fired)
    ge = np.sqrt(1 + sum(c * c for c in o["el_p"]))
    gp = np.sqrt(1 + sum(c * c for c in o["po_p"]))
    assert np.allclose(ge + gp, g[fired], rtol=1e-12)
    assert np.allclose(ge, 1 + (g[fired] - 2) * o["xi_el"], rtol=1e-12)
    assert np.all((o["xi_el"] >= 0) & (o["xi_el"] <= 1))
    for k in range(3):
        assert np.allclose(o["el_p"][k] / np.sqrt(ge ** 2 - 1), p[k][fired] / g[fired], atol=1e-9)
    assert all(np.all(o["p"][k][fired] == 0) for k in range(3)) and np.all(np.isinf(o["tau"][fired]))
    # electron <-> positron symmetry: r <= 1/2 gives the electron the smaller share
    r = np.array([orc.uniform(9, int(i), 4, 1, PHOTON, 0, F64) for i in fired])
    assert np.all((o["xi_el"] <= 0.5) == (r <= 0.5))
    assert abs(o["xi_el"].mean() - 0.5) < 4 * o["xi_el"].std() / math.sqrt(fired.size)


def test_capacity_rule(orc, small_tables):
    rng = np.random.default_rng(3)
    n = 200
    p, e, b, g = _population(rng, n, LEPTON)
    tau = np.where(np.arange(n) % 3 == 0, -0.5, 0.5)
    full = orc.generate_photons(small_tables, F64, F64, p, e, b, tau, 1, 0)
    part = orc.generate_photons(small_tables, F64, F64, p, e, b, tau, 1, 0, capacity=10)
    assert part["n_fired"] == full["n_fired"] == 67 and part["parent"].size == 10
    assert np.array_equal(part["parent"], full["parent"][:10])
    assert np.array_equal(part["ph_p"][0], full["ph_p"][0][:10])
    late = full["parent"][10:]
    assert np.all(part["tau"][late] == -0.5) and np.array_equal(part["p"][0][late], p[0][late])


def test_inverse_cdf_against_exact_cdf(orc):
    """eqs.24-26 / 28-30 on an oracle-built row reproduce the quantiles of the exact CDFs
    (eq.11 / eq.18 as the number CDF, R4) up to the table's interpolation error"""
    p = orc.TableParams(qs_chi_min=0.5, qs_chi_max=2.0, qs_n_chi=3, qs_xi_min=1e-12, qs_n_xi=193,
                        bw_chi_min=0.5, bw_chi_max=2.0, bw_n_chi=3, bw_n_xi=129)
    t = orc.build_tables(p)
    for r in (0.003, 0.1, 0.5, 0.9, 0.999):
        xi = orc.qs_sample_xi(t, 1.0, r)
        assert orc.qs_cdf(1.0, xi) == pytest.approx(r, rel=2e-3)
    for r in (0.01, 0.1, 0.3, 0.5):
        xi = orc.bw_sample_xi(t, 1.0, r)
        assert orc.bw_cdf(1.0, xi) == pytest.approx(r, rel=2e-3)
    # between rows: monotone in r, continuous across the bracket boundary chi = 1 (row 1)
    xs = [orc.qs_sample_xi(t, c, 0.37) for c in (0.999999, 1.0, 1.000001)]
    assert xs[0] == pytest.approx(xs[1], rel=1e-5) and xs[2] == pytest.approx(xs[1], rel=1e-5)
    # mean photon energy fraction under the number CDF at chi = 1 (0.117402)
    rs = (np.arange(20000) + 0.5) / 20000
    assert np.mean([orc.qs_sample_xi(t, 1.0, r) for r in rs]) == pytest.approx(0.117402, rel=5e-3)
    # below the first column: xi = xi_min (R6, unpinned by the paper)
    assert orc.qs_sample_xi(t, 1.0, 1e-9) == 1e-12


def test_inverse_cdf_closed_form_tables(orc):
    """with P = xi^{1/3} (QS) and P = xi (BW) stored exactly, the log-log / linear inverse
    interpolation is exact: xi = r^3 and xi = r'"""
    t = _power_law_tables(orc)
    for r in (1e-1, 0.3, 0.77, 0.999):
        assert orc.qs_sample_xi(t, 0.5, r) == pytest.approx(r ** 3, rel=1e-13)
    assert orc.qs_sample_xi(t, 0.5, 1e-3) == 1e-6      # r < P(xi_min) = 1e-2
    for r in (0.0, 0.01, 0.26, 0.5):
        assert orc.bw_sample_xi(t, 3.0, r) == pytest.approx(r, abs=1e-15)


def _row_dependent_tables(orc):
    """closed-form CDF tables whose rows DEPEND on chi: QS ln P[n][m] = a_n ln xi_m and BW P[n][m] = (2 xi_m)^2 (c_n +
    (1/2 - c_n) (2 xi_m)), with a_n and c_n linear in ln chi_n.  Interpolating the rows linearly in ln chi (PAPER.md:214
    eq.24, :257 eq.28) then gives exactly a(chi) ln xi and the same polynomial with c(chi), at any chi between rows."""
    p = orc.TableParams(qs_chi_min=1e-2, qs_chi_max=1e2, qs_n_chi=5, qs_xi_min=1e-6, qs_n_xi=13,
                        bw_chi_min=1e-1, bw_chi_max=1e3, bw_n_chi=5, bw_n_xi=9)
    lq = np.linspace(math.log(p.qs_chi_min), math.log(p.qs_chi_max), p.qs_n_chi)
    lb = np.linspace(math.log(p.bw_chi_min), math.log(p.bw_chi_max), p.bw_n_chi)
    a_of = lambda lc: 0.25 + 0.05 * (lc - lq[0])           # 0.25 .. 0.71 over the table
    c_of = lambda lc: 0.05 + 0.04 * (lc - lb[0])           # 0.05 .. 0.42
    lxi = math.log(p.qs_xi_min) * (1 - np.arange(p.qs_n_xi) / (p.qs_n_xi - 1))
    qs = np.outer(a_of(lq), lxi)
    u = 2 * (0.5 * np.arange(p.bw_n_xi) / (p.bw_n_xi - 1))
    bw = np.array([u * u * (c + (0.5 - c) * u) for c in c_of(lb)])
    return orc.Tables(p, np.zeros(p.qs_n_chi), qs, np.zeros(p.bw_n_chi), bw), a_of, c_of


def test_row_interpolation_weight_is_linear_in_ln_chi(orc):
    """the weight of eq.24 / eq.28 between rows n and n+1 is (ln chi - ln chi_n)/(ln chi_{n+1} - ln chi_n)
    (PAPER.md:214, :257): a weight linear in chi itself gives another row and fails these closed forms"""
    t, a_of, c_of = _row_dependent_tables(orc)
    # QS: interpolated row = a(chi) ln xi  =>  eq.30 (log-log, exact for a power law) gives xi = r^{1/a(chi)}
    for chi in (0.013, 0.3, 1.0, 2.7, 31.0, 88.0):           # strictly between rows (rows at 1e-2, 1e-1, 1, 10, 100)
        a = a_of(math.log(chi))
        for r in (0.05, 0.4, 0.93):
            if r > 1e-6 ** a:                                 # above the first column
                assert orc.qs_sample_xi(t, chi, r) == pytest.approx(r ** (1 / a), rel=1e-12)
    # the mid-point in ln chi between two rows, against the mid-point in chi (which must NOT be what is used)
    lo, hi = 1.0, 10.0
    chi_geo, a_geo = math.sqrt(lo * hi), 0.5 * (a_of(math.log(lo)) + a_of(math.log(hi)))
    assert orc.qs_sample_xi(t, chi_geo, 0.4) == pytest.approx(0.4 ** (1 / a_geo), rel=1e-12)
    assert orc.qs_sample_xi(t, 0.5 * (lo + hi), 0.4) != pytest.approx(0.4 ** (1 / a_geo), rel=1e-3)
    # BW: interpolated row = u^2 (c + (1/2 - c) u), u = 2 xi, c = c(chi) linear in ln chi; eq.26 interpolates linearly
    # between columns, so compare at the table's own columns where that is exact: r' = P(xi_m) -> xi_m
    for chi in (0.17, 3.3, 40.0, 700.0):
        c = c_of(math.log(chi))
        for m in (2, 5, 7):
            xi_m = 0.5 * m / 8
            u = 2 * xi_m
            assert orc.bw_sample_xi(t, chi, u * u * (c + (0.5 - c) * u)) == pytest.approx(xi_m, abs=1e-13)
        # and inside a cell: the linear inverse of the two bracketing columns of THAT interpolated row
        u0, u1 = 2 * 0.5 * 4 / 8, 2 * 0.5 * 5 / 8
        P0, P1 = u0 * u0 * (c + (0.5 - c) * u0), u1 * u1 * (c + (0.5 - c) * u1)
        rp = 0.3 * P0 + 0.7 * P1
        assert orc.bw_sample_xi(t, chi, rp) == pytest.approx(0.5 * (4 + 0.7) / 8, abs=1e-13)


def test_row_interpolation_on_a_row_grid_of_its_own(orc):
    """2D tables whose rows sit on another chi grid than the 1D tables (BASELINE config 4: 4096 and 2048 points): the
    row bracket uses the 2D grid -- the same closed forms hold with 9 (QS) / 7 (BW) 1D points over 5 rows"""
    t, a_of, c_of = _row_dependent_tables(orc)
    p = orc.TableParams(**dict(t.params.__dict__, qs_n_chi=9, bw_n_chi=7, qs_n_chi_2d=5, bw_n_chi_2d=5))
    t2 = orc.Tables(p, np.zeros(9), t.qs_lnP, np.zeros(7), t.bw_P)
    for chi in (0.013, 2.7, 31.0):
        assert orc.qs_sample_xi(t2, chi, 0.4) == pytest.approx(0.4 ** (1 / a_of(math.log(chi))), rel=1e-12)
        assert orc.qs_sample_xi(t2, chi, 0.4) == orc.qs_sample_xi(t, chi, 0.4)
    for chi in (0.17, 40.0):
        assert orc.bw_sample_xi(t2, chi, 0.21) == orc.bw_sample_xi(t, chi, 0.21)


def test_row_interpolation_between_rows_of_a_built_table(orc):
    """at chi strictly between two closely spaced rows of an oracle-built table, the sampled xi has the exact CDF
    value r (eq.11 / eq.18 by quadrature at THAT chi) up to the interpolation error of the table"""
    p = orc.TableParams(qs_chi_min=0.8, qs_chi_max=1.25, qs_n_chi=3, qs_xi_min=1e-12, qs_n_xi=193,
                        bw_chi_min=0.8, bw_chi_max=1.25, bw_n_chi=3, bw_n_xi=129)
    t = orc.build_tables(p)
    for chi in (0.9, 1.1):                                     # rows at 0.8, 1.0, 1.25
        for r in (0.1, 0.5, 0.9):
            assert orc.qs_cdf(chi, orc.qs_sample_xi(t, chi, r)) == pytest.approx(r, rel=2e-3)
        for r in (0.1, 0.3, 0.5):
            assert orc.bw_cdf(chi, orc.bw_sample_xi(t, chi, r)) == pytest.approx(r, rel=2e-3)


def _stream_uniform(orc, seed, pid, step, purpose, species, pair):
    """the documented stream, typed out here: key = (seed_lo, seed_hi),
    counter = (id_lo, id_hi, step_lo, purpose | species << 8 | step_hi16 << 16); words (2 pair, 2 pair + 1) -> the top
    52 bits + 1/2, times 2^-52.  Only the block function comes from the oracle (pinned by the published vectors)."""
    ctr = (pid & 0xFFFFFFFF, pid >> 32, step & 0xFFFFFFFF, purpose | (species << 8) | (((step >> 32) & 0xFFFF) << 16))
    w = orc.philox4x32_10(ctr, (seed & 0xFFFFFFFF, seed >> 32))
    k = ((w[2 * pair] << 32) | w[2 * pair + 1]) >> 12
    return (k + 0.5) * 2.0 ** -52


def test_children_and_parent_streams(orc, small_tables):
    """purpose 1 words (2,3): the parent's new optical depth; purpose 2 words (0,1): photon / electron, words (2,3):
    positron -- so the two members of a pair are born with DIFFERENT optical depths"""
    rng = np.random.default_rng(11)
    n, seed, step, base = 400, 77, (3 << 32) | 5, 1 << 40
    ids = base + np.arange(n, dtype=np.uint64)
    tau = np.where(rng.random(n) < 0.5, -rng.random(n), rng.random(n) + 0.1)
    p, e, b, _ = _population(rng, n, LEPTON)
    o = orc.generate_photons(small_tables, F64, F64, p, e, b, tau, seed, step, ids=ids)
    for slot, i in enumerate(o["parent"]):
        pid = base + int(i)
        assert o["tau"][i] == pytest.approx(-math.log(_stream_uniform(orc, seed, pid, step, 1, LEPTON, 1)), rel=1e-15)
        assert o["ph_tau"][slot] == pytest.approx(-math.log(_stream_uniform(orc, seed, pid, step, 2, LEPTON, 0)), rel=1e-15)
    p, e, b, _ = _population(rng, n, PHOTON)
    o = orc.generate_pairs(small_tables, F64, F64, p, e, b, tau, seed, step, ids=ids)
    assert o["n_fired"] > 100
    for slot, i in enumerate(o["parent"]):
        pid = base + int(i)
        assert o["el_tau"][slot] == pytest.approx(-math.log(_stream_uniform(orc, seed, pid, step, 2, PHOTON, 0)), rel=1e-15)
        assert o["po_tau"][slot] == pytest.approx(-math.log(_stream_uniform(orc, seed, pid, step, 2, PHOTON, 1)), rel=1e-15)
    assert np.all(o["el_tau"] != o["po_tau"])
    # and the oracle's own orc_uniform helper follows the same layout (it is what the GPU tests call)
    assert orc.uniform(seed, base + 9, step, 2, PHOTON, 1, F64) == _stream_uniform(orc, seed, base + 9, step, 2, PHOTON, 1)


# ----------------------------------------------------------------------------- chi threshold and classical model
def test_chi_threshold_switches_both_processes_off(orc):
    """below the threshold neither process is an event: the rate is exactly 0, at and above it the rate is unchanged"""
    t = _power_law_tables(orc)
    tt = t.with_chi_event_min(0.5)
    for sp, pm in ((LEPTON, 1000.0), (PHOTON, 500.0)):
        for chi_want, below in ((0.2, True), (0.4999, True), (0.5001, False), (7.0, False)):
            args = (vec((pm, 0, 0)), vec((0, 0, 0)), vec((0, chi_want / pm, 0)))
            r0, r1 = orc.rate(t, sp, *args)[0], orc.rate(tt, sp, *args)[0]
            assert r0 > 0 and (r1 == 0.0 if below else r1 == r0)
    # evolve: optical depths of the particles below the threshold do not move
    n = 1000
    rng = np.random.default_rng(5)
    p, e, b, g = _population(rng, n, LEPTON)
    chi = orc.chi(LEPTON, p, e, b)
    tau = rng.exponential(size=n)
    o = orc.evolve_optical_depth(tt, LEPTON, F64, p, e, b, 1e-15, tau)
    assert np.array_equal(o["tau"][chi < 0.5], tau[chi < 0.5]) and np.all(o["tau"][chi >= 0.5] < tau[chi >= 0.5])


def test_classical_loss_closed_form_and_bookkeeping(orc):
    """p perp b: chi = |p||b|; one step removes (2/3)(alpha/tau_C) chi^2 (gamma-1)/gamma dt of kinetic energy, keeps the
    direction, leaves the leptons at or above the threshold alone and never takes the kinetic energy below zero"""
    pm, bb, dt = 300.0, 1e-6, 2e-13
    g = math.sqrt(1 + pm * pm)
    chi = pm * bb
    p2 = orc.classical_loss(F64, vec((0, pm, 0)), vec((0, 0, 0)), vec((bb, 0, 0)), dt, 1e-3)
    k_after = math.sqrt(1 + p2[1][0] ** 2) - 1
    want = (g - 1) - 2 / 3 * ALPHA_OVER_TAUC * chi * chi * (g - 1) / g * dt
    assert p2[0][0] == 0 and p2[2][0] == 0 and p2[1][0] > 0
    assert k_after == pytest.approx(want, rel=1e-12) and 0 < 1 - want / (g - 1) < 0.5
    # at / above the threshold: untouched, bit for bit
    same = orc.classical_loss(F64, vec((0, pm, 0)), vec((0, 0, 0)), vec((bb, 0, 0)), dt, chi)
    assert same[1][0] == pm
    # a step that would take more than there is stops at rest
    rest = orc.classical_loss(F64, vec((0, pm, 0)), vec((0, 0, 0)), vec((bb, 0, 0)), 1e-6, 1e-3)
    assert rest[1][0] == 0.0
    # a random population: direction kept, energy never gained, fp32 storage rounds once
    rng = np.random.default_rng(8)
    p, e, b, g = _population(rng, 500, LEPTON)
    chi = orc.chi(LEPTON, p, e, b)
    q = orc.classical_loss(F64, p, e, b, 1e-16, 0.05)
    low = chi < 0.05
    assert 0 < low.sum() < 500 and all(np.array_equal(a[~low], c[~low]) for a, c in zip(p, q))
    n0, n1 = np.sqrt(sum(a * a for a in p)), np.sqrt(sum(a * a for a in q))
    assert np.all(n1[low] < n0[low])
    for a, c in zip(p, q):
        assert np.allclose(c[low] / n1[low], a[low] / n0[low], atol=1e-13)
    q32 = orc.classical_loss(F32, p, e, b, 1e-16, 0.05)
    assert all(np.array_equal(c[low], c[low].astype(np.float32).astype(np.float64)) for c in q32)


def test_classical_loss_is_the_small_chi_limit_of_the_mean_emission(orc):
    """continuity across the threshold: the mean energy a lepton loses per unit time to the Monte Carlo emission,
    rate x (gamma-1) x <xi> with <xi> = int S dxi / G (exact quadratures), tends to the classical power as chi -> 0"""
    pm, dt = 2000.0, 1e-18
    g = math.sqrt(1 + pm * pm)
    for chi, tol in ((1e-3, 1e-2), (1e-2, 6e-2)):        # the quantum correction is 1 - 5.95 chi + ...
        mc = 2 / 3 * ALPHA_OVER_TAUC * orc.qs_first_moment(chi) * (g - 1) / g          # rate x <xi> x (gamma-1), G cancels
        p2 = orc.classical_loss(F64, vec((0, pm, 0)), vec((0, 0, 0)), vec((chi / pm, 0, 0)), dt, 1.0)
        cl = ((g - 1) - (math.sqrt(1 + p2[1][0] ** 2) - 1)) / dt
        assert cl == pytest.approx(2 / 3 * ALPHA_OVER_TAUC * chi * chi * (g - 1) / g, rel=1e-6)
        assert mc < cl and mc == pytest.approx(cl, rel=tol)


# ----------------------------------------------------------------------------- Schwinger rate
def test_schwinger_rate_closed_forms(orc):
    """PAPER.md:171-183 eqs.19-22: prefactor from CODATA, pure-E textbook limit, E parallel B, null fields"""
    hbar = 6.62607015e-34 / (2 * math.pi)
    m, c = 9.1093837015e-31, 299792458.0
    C = m ** 4 * c ** 5 / (4 * math.pi ** 2 * hbar ** 4)   # q^2 E_s^2/(4 pi^2 hbar^2 c) with E_s = m^2 c^3/(q hbar)
    assert orc.schwinger_prefactor() == pytest.approx(C, rel=1e-13)
    z = np.zeros(4)
    ev = np.array([1.0, 0.3, 0.1, 0.05])
    # pure electric field: (qE)^2/(4 pi^3 hbar^2 c) exp(-pi E_s/E), the leading term of Schwinger's formula
    r = orc.schwinger_rate([ev, z, z], [z, z, z])
    assert np.allclose(r, C * ev ** 2 / math.pi * np.exp(-math.pi / ev), rtol=1e-14)
    # E parallel B: epsilon = E/E_s, eta = cB/E_s exactly (F = (e^2-b^2)/2, G = e b)
    bv = np.array([0.5, 0.3, 0.02, 0.4])
    r = orc.schwinger_rate([z, ev, z], [z, bv, z])
    assert np.allclose(r, C * ev * bv / np.tanh(math.pi * bv / ev) * np.exp(-math.pi / ev), rtol=1e-13)
    # pure magnetic field, and a plane wave (e perpendicular to b, equal norms: F = G = 0): no pairs
    assert np.all(orc.schwinger_rate([z, z, z], [bv, z, z]) == 0)
    assert np.all(orc.schwinger_rate([ev, z, z], [z, ev, z]) == 0)
    # weak-field values are representable far below double underflow of exp(-pi/eps) * C? (C ~ 3e56)
    assert orc.schwinger_rate([np.array([0.005])] + [np.zeros(1)] * 2, [np.zeros(1)] * 3)[0] == pytest.approx(
        C * 0.005 ** 2 / math.pi * math.exp(-math.pi / 0.005), rel=1e-12)


def test_schwinger_rate_is_lorentz_invariant(orc):
    """the rate depends on the fields only through the invariants F and G: rotations, boosts, G -> -G"""
    rng = np.random.default_rng(11)
    n = 200
    e = rng.normal(size=(3, n)) * 0.3
    b = rng.normal(size=(3, n)) * 0.3
    r0 = orc.schwinger_rate(list(e), list(b))
    # rotation
    q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    assert np.allclose(orc.schwinger_rate(list(q @ e), list(q @ b)), r0, rtol=1e-12)
    # boost along x with velocity beta: parallel components unchanged, e_perp' = g (e + beta x b), b_perp' = g (b - beta x e)
    beta = 0.6
    g = 1 / math.sqrt(1 - beta * beta)
    e2 = np.array([e[0], g * (e[1] - beta * b[2]), g * (e[2] + beta * b[1])])
    b2 = np.array([b[0], g * (b[1] + beta * e[2]), g * (b[2] - beta * e[1])])
    assert np.allclose(orc.schwinger_rate(list(e2), list(b2)), r0, rtol=1e-11)
    # parity: b -> -b flips the sign of G only
    assert np.allclose(orc.schwinger_rate(list(e), list(-b)), r0, rtol=1e-13)
    assert np.all(r0 >= 0) and np.any(r0 > 0)
