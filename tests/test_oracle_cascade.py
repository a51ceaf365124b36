"""Pins of the closed-loop oracle (oracle/cascade.py) against what the mathematics and
the paper fix: closed forms of the Boris scheme, the published Compton wavelength, bookkeeping invariants of the
loop, and the quantum-corrected radiated power at chi = 1 (SURVEY.md App. B values) for Ridgers case (i)."""
import numpy as np
import pytest

from oracle import cascade as cas


def _rand_u(n, seed, scale=50.0):
    rng = np.random.default_rng(seed)
    return [scale * rng.standard_normal(n) for _ in range(3)]


def test_inv_tau_c_is_c_over_reduced_compton_wavelength(orc):
    # CODATA 2018 reduced Compton wavelength 3.8615926796(12)e-13 m: an independently published number
    assert abs(float(cas.inv_tau_c()) / (299792458.0 / 3.8615926796e-13) - 1) < 1e-9
    # and the oracle's own rate prefactor alpha m c^2/hbar (eq.8) with CODATA alpha
    assert abs(orc.rate_prefactor() / (7.2973525693e-3 * float(cas.inv_tau_c())) - 1) < 1e-9


def test_boris_pure_electric_field_is_a_linear_kick():
    u = _rand_u(1000, 1)
    e, dt = (3e-4, -2e-4, 5e-5), 1.7e-19
    for s in (-1, +1):
        un = cas.boris_push_uniform(u, s, e, (0, 0, 0), dt)
        for c in range(3):
            assert np.allclose(un[c], u[c] + s * e[c] * dt * float(cas.inv_tau_c()), rtol=1e-15, atol=1e-13)


def test_boris_rotation_closed_form_and_sense():
    """pure B: |u| is conserved, the component along b is untouched, and the perpendicular part turns by exactly
    theta = 2 atan(|b| dt/(2 tau_C gamma)) (textbook property of the scheme); an electron moving along +x in
    B = +z is pushed towards +y (F = q v x B, q < 0), a positron towards -y"""
    n = 2000
    u = _rand_u(n, 2)
    b = np.array([2e-4, -1e-4, 3e-4])
    dt = 4e-19
    g = np.sqrt(1 + sum(a * a for a in u))
    for s in (-1, +1):
        un = cas.boris_push_uniform(u, s, (0, 0, 0), b, dt)
        U, UN = np.stack(u), np.stack(un)
        assert np.allclose((UN * UN).sum(0), (U * U).sum(0), rtol=4e-16)
        bh = b / np.linalg.norm(b)
        assert np.allclose(bh @ UN, bh @ U, rtol=1e-13, atol=1e-13)
        perp, perpn = U - np.outer(bh, bh @ U), UN - np.outer(bh, bh @ UN)
        cosang = (perp * perpn).sum(0) / (perp * perp).sum(0)
        theta = 2 * np.arctan(np.linalg.norm(b) * dt * float(cas.inv_tau_c()) / (2 * g))
        assert np.allclose(np.arccos(np.clip(cosang, -1, 1)), theta, rtol=1e-9)
        # sense: d u/dt = s (u/gamma) x b / tau_C
        sense = np.sign((np.cross(perp.T, perpn.T) @ bh))
        assert np.all(sense == -s)
    one = cas.boris_push_uniform([np.array([10.0]), np.array([0.0]), np.array([0.0])], -1, (0, 0, 0), (0, 0, 1e-3), 1e-19)
    assert one[1][0] > 0
    one = cas.boris_push_uniform([np.array([10.0]), np.array([0.0]), np.array([0.0])], +1, (0, 0, 0), (0, 0, 1e-3), 1e-19)
    assert one[1][0] < 0


def test_boris_converges_to_the_analytic_gyration_at_second_order():
    """gamma is constant in pure B, so the exact motion is a rotation by omega T, omega = |b|/(tau_C gamma); the
    scheme's phase error is O(dt^2): halving dt divides it by 4"""
    u0 = [np.array([1000.0]), np.array([0.0]), np.array([0.0])]
    b = (0.0, 0.0, 1e-3)
    gam = np.sqrt(1 + 1000.0 ** 2)
    T = 2e-17
    exact_angle = 1e-3 * float(cas.inv_tau_c()) * T / gam
    errs = []
    for nst in (50, 100, 200):
        u = u0
        for _ in range(nst):
            u = cas.boris_push_uniform(u, +1, (0, 0, 0), b, T / nst)
        ang = np.arctan2(-u[1][0], u[0][0])  # positron turns clockwise seen from +z
        errs.append(abs(ang - exact_angle))
    assert errs[0] < 1e-3 * exact_angle
    assert 3.6 < errs[0] / errs[1] < 4.4 and 3.6 < errs[1] / errs[2] < 4.4


def test_boris_parallel_fields_decouple():
    """e parallel to b: the momentum along the field grows linearly in time whatever the gyration does"""
    u = _rand_u(500, 3, scale=5.0)
    axis = np.array([1.0, 2.0, -2.0]) / 3.0
    e, b = 2e-4 * axis, 7e-4 * axis
    dt, nst = 3e-19, 40
    v = u
    for _ in range(nst):
        v = cas.boris_push_uniform(v, -1, e, b, dt)
    par0, par1 = axis @ np.stack(u), axis @ np.stack(v)
    assert np.allclose(par1, par0 - 2e-4 * nst * dt * float(cas.inv_tau_c()), rtol=1e-12, atol=1e-12)


def test_energy_spectrum_bins_and_exclusions(orc):
    nb, lo, hi = 12, 1e-2, 1e4
    edges = np.exp(np.linspace(np.log(lo), np.log(hi), nb + 1))
    centres = np.sqrt(edges[:-1] * edges[1:])
    # photons: |p| at the bin centres, k+1 copies in bin k, plus dead, below-range and above-range entries
    en = np.concatenate([np.repeat(centres, np.arange(1, nb + 1)), [0.0, 0.0, 1e-3, 5e4, hi]])
    rng = np.random.default_rng(5)
    d = rng.standard_normal((3, en.size))
    d /= np.linalg.norm(d, axis=0)
    h, _ = cas.energy_spectrum(orc.PHOTON, list(d * en), lo, hi, nb)
    assert h.tolist() == list(range(1, nb + 1))
    # leptons: kinetic energy gamma - 1, from p = sqrt(gamma^2 - 1)
    gam = 1 + np.repeat(centres, 2)
    pl = np.sqrt(gam * gam - 1)
    h, x = cas.energy_spectrum(orc.LEPTON, [pl, 0 * pl, 0 * pl], lo, hi, nb)
    assert h.tolist() == [2] * nb and np.allclose(x - np.floor(x), 0.5, atol=1e-6)


@pytest.fixture(scope="module")
def chi1_tables(orc):
    """photon-emission tables in a narrow band around chi = 1, fine in xi (a few seconds)"""
    p = orc.TableParams(qs_chi_min=0.5, qs_chi_max=2.0, qs_n_chi=9, qs_xi_min=1e-12, qs_n_xi=193,
                        bw_chi_min=0.5, bw_chi_max=2.0, bw_n_chi=5, bw_n_xi=17)
    return orc.build_tables(p)


def _case_i(orc, n, seed):
    """Ridgers case (i): gamma_0 = 1000, perpendicular static B_0 = 1e-3 E_s/c, chi = 1"""
    g0 = 1000.0
    p0 = np.sqrt(g0 * g0 - 1)
    el = cas.Population([np.full(n, p0), np.zeros(n), np.zeros(n)],
                        orc.init_optical_depth(orc.LEPTON, orc.F64, n, seed, np.arange(n, dtype=np.uint64)))
    return {"electrons": el, "positrons": cas.empty_population(), "photons": cas.empty_population()}, g0


def test_case_i_initial_chi_is_one(orc):
    pops, g0 = _case_i(orc, 4, 1)
    n = 4
    chi = orc.chi(orc.LEPTON, pops["electrons"].p, [np.zeros(n)] * 3, [np.zeros(n), np.zeros(n), np.full(n, 1e-3)])
    assert np.allclose(chi, np.sqrt(g0 * g0 - 1) * 1e-3, rtol=1e-12)   # PAPER.md:346 "initial quantum parameter chi = 1"


def test_case_i_mean_energy_loss_matches_the_quantum_radiated_power(orc, chi1_tables):
    """closed loop over 10 steps (push, evolve, emission, feedback): the mean energy lost per electron must be
    rate * <xi> * (gamma - 1) * T with rate = (2/3)(alpha/tau_C) G(chi)/gamma (eq.15) and the values of
    SURVEY.md App. B at chi = 1: G = 1.550870924, <xi> = 0.117402.  About 2e4 events: sigma = 1.3 %; chi drifts by
    0.6 % during the run.  Every photon that is emitted is fed back and carries exactly the energy its emitter lost."""
    n, steps = 400_000, 10
    pops, g0 = _case_i(orc, n, 11)
    rate = (2.0 / 3.0) * orc.rate_prefactor() * 1.550870924 / g0
    dt = 0.05 / rate / steps
    e, b = (0.0, 0.0, 0.0), (0.0, 0.0, 1e-3)
    events = 0
    for s in range(steps):
        r = cas.cascade_step(chi1_tables, orc.F64, orc.F64, pops, e, b, dt, 11, s)
        events += r["events"][0]
        assert r["events"][1] == 0 and r["photons_kept"] == r["events"][0]
    el, ph = pops["electrons"], pops["photons"]
    assert el.n == n and ph.n == events and pops["positrons"].n == 0
    gam = np.sqrt(1 + sum(a * a for a in el.p))
    lost = g0 - gam.mean()
    expect = rate * 0.117402 * (g0 - 1) * dt * steps
    assert abs(events / n / 0.05 - 1) < 0.04           # 1 - exp(-R dt) summed, R falling slowly
    assert abs(lost / expect - 1) < 0.05, (lost, expect)
    # energy bookkeeping of the loop: what the electrons lost is what the photons carry
    eph = np.sqrt(sum(a * a for a in ph.p)).sum()
    assert abs(eph / (n * lost) - 1) < 1e-9
    # the photons fly along the (rotated) momenta: all in the plane perpendicular to b
    assert np.all(ph.p[2] == 0) and np.all(el.p[2] == 0)


def test_photon_threshold_discards_the_photon_but_debits_the_emitter(orc, chi1_tables):
    """below the threshold "the emitting particle is slowed down as if the photon were emitted, but the
    photon particle is discarded immediately after creation" (strict <, R22)"""
    n = 20_000
    e, b = (0.0, 0.0, 0.0), (0.0, 0.0, 1e-3)
    rate = (2.0 / 3.0) * orc.rate_prefactor() * 1.550870924 / 1000.0
    runs = {}
    for thr in (0.0, 2.0, np.inf):
        pops, g0 = _case_i(orc, n, 12)
        r = cas.cascade_step(chi1_tables, orc.F64, orc.F64, pops, e, b, 0.3 / rate, 12, 0, photon_min_energy=thr)
        runs[thr] = (pops, r)
    (p0, r0), (p2, r2), (pinf, rinf) = runs[0.0], runs[2.0], runs[np.inf]
    assert r0["events"] == r2["events"] == rinf["events"] and r0["events"][0] > 1000
    for c in range(3):   # the emitters are debited identically in all three runs
        assert np.array_equal(p0["electrons"].p[c], p2["electrons"].p[c])
        assert np.array_equal(p0["electrons"].p[c], pinf["electrons"].p[c])
    assert pinf["photons"].n == 0 and p0["photons"].n == r0["events"][0]
    g_all = np.sqrt(sum(a * a for a in p0["photons"].p))
    keep = g_all >= 2.0
    assert 0 < keep.sum() < g_all.size and p2["photons"].n == keep.sum()
    for c in range(3):   # the survivors keep their order
        assert np.array_equal(p2["photons"].p[c], p0["photons"].p[c][keep])
    assert np.array_equal(p2["photons"].tau, p0["photons"].tau[keep])


def test_cascade_case_iii_feeds_pairs_back_with_unique_ids(orc, small_tables):
    """Ridgers case (iii): gamma_0 = 1000 in B_0 = 9e-3 E_s/c (chi = 9): photons decay, pairs join the
    lepton arrays and radiate in turn.  Bookkeeping invariants of the loop: arrays only grow, every decayed photon is
    a dead entry (R21) and gave one electron and one positron, and total energy (kinetic + 1 per lepton, photons at
    face value) is conserved by every event."""
    n, steps = 3000, 30
    g0 = 1000.0
    p0 = np.sqrt(g0 * g0 - 1)
    el = cas.Population([np.full(n, p0), np.zeros(n), np.zeros(n)], orc.init_optical_depth(orc.LEPTON, orc.F64, n, 13))
    pops = {"electrons": el, "positrons": cas.empty_population(), "photons": cas.empty_population()}
    e, b = (0.0, 0.0, 0.0), (0.0, 0.0, 9e-3)
    dt = 1e-16 / steps   # 0.1 fs
    n_pairs = 0
    for s in range(steps):
        before = {k: v.n for k, v in pops.items()}
        r = cas.cascade_step(small_tables, orc.F64, orc.F64, pops, e, b, dt, 13, s)
        n_pairs += r["events"][2]
        assert pops["electrons"].n == before["electrons"] + r["events"][2]
        assert pops["positrons"].n == before["positrons"] + r["events"][2]
        assert pops["photons"].n == before["photons"] + r["events"][0] + r["events"][1]
    assert n_pairs > 20
    ph = pops["photons"]
    dead = (ph.p[0] == 0) & (ph.p[1] == 0) & (ph.p[2] == 0)
    assert dead.sum() == n_pairs and np.all(np.isinf(ph.tau[dead])) and np.all(np.isfinite(ph.tau[~dead]))
    energy = lambda pop: np.sqrt(1 + sum(a * a for a in pop.p)).sum()
    total = energy(pops["electrons"]) + energy(pops["positrons"]) + np.sqrt(sum(a * a for a in ph.p)).sum()
    assert abs(total / (n * g0) - 1) < 1e-9   # pure B does no work; every event conserves energy (R15)
