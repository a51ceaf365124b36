"""Closed loop in a uniform field -- oracle.  TEST INFRASTRUCTURE, NOT THE PRODUCT.

SURVEY.md 8(f)-1 and 8(f)-2: the Ridgers test cases (i) and (iii) the paper reproduces with WarpX
(an electron population of Lorentz factor gamma_0 in a perpendicular, static,
uniform magnetic field), run with the library's own QED step: leptons are pushed, every species
takes its QED step, secondaries are fed back, photons below an energy threshold are
discarded right after creation while the emitter is still slowed down, and the
energy spectra of Fig.6 are histogrammed.

Plain numpy, fp64 (the pusher in long double), one statement per formula, no blocking or reordering.
Units: momenta in m_e c, energies in m_e c^2, e = E/E_s, b = cB/E_s, times in seconds.

Readings (R19-R23), the paper being silent on all of them:
  R19 pusher: the standard Boris scheme (half electric kick, magnetic rotation with
      t = s b dt/(2 tau_C gamma^-), second half kick), s = -1 electron, +1 positron; in these units
      du/dt = s (e + (u/gamma) x b)/tau_C, tau_C = hbar/(m_e c^2).
  R20 order inside a time step: push the leptons -> QED step of electrons, positrons, photons on the
      populations that existed when the step began -> append the secondaries (photons of the
      electrons first, then those of the positrons).  A particle takes no part in the step that
      created it.
  R21 a photon that decayed stays in its array as a dead entry (p = 0, tau = +inf, R12);
      array positions never change, so the Philox id of a particle (id_base of its array + position)
      is fixed for its lifetime.
  R22 photon threshold: a new photon with gamma_gamma = |p| < photon_min_energy is not appended
      (strict <, "below such threshold").
  R23 spectrum: histogram over nbins logarithmic bins of [e_min, e_max) of the kinetic energy
      gamma - 1 = p^2/(gamma + 1) (leptons; this form does not cancel) or gamma_gamma = |p| (photons);
      bin = floor((ln E - ln e_min) nbins/(ln e_max - ln e_min)) in fp64; dead entries (p = 0) and
      energies outside the range are not counted.
"""
import numpy as np

from . import api

# CODATA 2018 (exact c, h; recommended m_e), typed here independently of the CUDA side
_C = 299792458.0
_H = 6.62607015e-34
_ME = 9.1093837015e-31

ID_BASE = {"electrons": 0, "positrons": 1 << 40, "photons": 1 << 41}


def inv_tau_c():
    """m_e c^2 / hbar [1/s]: the rate at which a field e = 1 changes u = p/(m_e c) (R19)"""
    L = np.longdouble
    return L(_ME) * L(_C) * L(_C) * (2 * np.pi * L(1)) / L(_H)


def boris_push_uniform(p, sign, e, b, dt):
    """R19, step by step in long double.  p: three arrays; e, b: three numbers each; returns three fp64 arrays"""
    L = np.longdouble
    u = np.stack([np.asarray(a, dtype=np.float64).astype(L) for a in p])          # (3, n)
    ev = np.array(e, dtype=np.float64).astype(L).reshape(3, 1)
    bv = np.array(b, dtype=np.float64).astype(L).reshape(3, 1)
    k = L(sign) * L(dt) * inv_tau_c() / 2                                           # s dt / (2 tau_C)
    um = u + k * ev                                                                 # half electric kick
    gm = np.sqrt(1 + (um * um).sum(axis=0))                                         # gamma^-
    t = k * bv / gm                                                                 # rotation vector
    up = um + np.cross(um, t, axis=0)                                               # u' = u^- + u^- x t
    s = 2 * t / (1 + (t * t).sum(axis=0))
    uplus = um + np.cross(up, s, axis=0)                                            # u^+ = u^- + u' x s
    un = uplus + k * ev                                                             # second half kick
    return [un[c].astype(np.float64) for c in range(3)]


def energy_spectrum(species, p, e_min, e_max, nbins):
    """R23.  Returns (hist[nbins] int64, position in bin units (float, nan where not counted))"""
    px, py, pz = [np.asarray(a, dtype=np.float64) for a in p]
    p2 = px * px + py * py + pz * pz
    if species == api.LEPTON:
        en = p2 / (np.sqrt(1 + p2) + 1)
    else:
        en = np.sqrt(p2)
    live = p2 > 0
    with np.errstate(divide="ignore", invalid="ignore"):
        x = (np.log(en) - np.log(e_min)) * (nbins / (np.log(e_max) - np.log(e_min)))
    x = np.where(live, x, np.nan)
    ok = live & (x >= 0) & (x < nbins)
    hist = np.bincount(np.floor(x[ok]).astype(np.int64), minlength=nbins).astype(np.int64)
    return hist, np.where(ok, x, np.nan)


class Population:
    """one species: structure of arrays, entries [0, n) in use"""

    def __init__(self, p, tau):
        self.p = [np.array(a, dtype=np.float64) for a in p]
        self.tau = np.array(tau, dtype=np.float64)

    @property
    def n(self):
        return self.tau.size

    def append(self, p, tau):
        self.p = [np.concatenate([a, np.asarray(c, dtype=np.float64)]) for a, c in zip(self.p, p)]
        self.tau = np.concatenate([self.tau, np.asarray(tau, dtype=np.float64)])


def empty_population():
    return Population([np.zeros(0)] * 3, np.zeros(0))


def keep_photons(ph_p, photon_min_energy):
    """R22: mask of the new photons that are appended"""
    g = np.sqrt(ph_p[0] ** 2 + ph_p[1] ** 2 + ph_p[2] ** 2)
    return ~(g < photon_min_energy)


def qed_step_species(tables, species, dtype, tau_dtype, pop, e, b, dt, seed, step, id_base):
    """evolve + events of one species in the uniform field (e, b); returns the event dict"""
    n = pop.n
    ee = [np.full(n, float(v)) for v in e]
    bb = [np.full(n, float(v)) for v in b]
    ids = np.uint64(id_base) + np.arange(n, dtype=np.uint64)
    tau = api.evolve_optical_depth(tables, species, tau_dtype, pop.p, ee, bb, dt, pop.tau)["tau"]
    if species == api.LEPTON:
        o = api.generate_photons(tables, dtype, tau_dtype, pop.p, ee, bb, tau, seed, step, ids)
    else:
        o = api.generate_pairs(tables, dtype, tau_dtype, pop.p, ee, bb, tau, seed, step, ids)
    pop.p, pop.tau = o["p"], o["tau"]
    return o


def cascade_step(tables, dtype, tau_dtype, pops, e, b, dt, seed, step, photon_min_energy=0.0, push=True):
    """one time step in the order of R20.  pops: dict electrons / positrons / photons -> Population (modified).
    Returns the numbers of events (electrons, positrons, photons) and of photons kept.
    With tables.chi_event_min > 0 (R24) the leptons below the threshold take one step of the classical
    radiation reaction after the push, and no particle below it has an event."""
    el, po, ph = pops["electrons"], pops["positrons"], pops["photons"]
    if push:
        el.p = boris_push_uniform(el.p, -1, e, b, dt)
        po.p = boris_push_uniform(po.p, +1, e, b, dt)
        if dtype == api.F32:
            el.p = [a.astype(np.float32).astype(np.float64) for a in el.p]
            po.p = [a.astype(np.float32).astype(np.float64) for a in po.p]
    if tables.chi_event_min > 0:
        for pop in (el, po):
            ee = [np.full(pop.n, float(v)) for v in e]
            bb = [np.full(pop.n, float(v)) for v in b]
            pop.p = api.classical_loss(dtype, pop.p, ee, bb, dt, tables.chi_event_min)
    oe = qed_step_species(tables, api.LEPTON, dtype, tau_dtype, el, e, b, dt, seed, step, ID_BASE["electrons"])
    op = qed_step_species(tables, api.LEPTON, dtype, tau_dtype, po, e, b, dt, seed, step, ID_BASE["positrons"])
    og = qed_step_species(tables, api.PHOTON, dtype, tau_dtype, ph, e, b, dt, seed, step, ID_BASE["photons"])
    kept = 0
    for o in (oe, op):
        m = keep_photons(o["ph_p"], photon_min_energy)
        ph.append([a[m] for a in o["ph_p"]], o["ph_tau"][m])
        kept += int(m.sum())
    el.append(og["el_p"], og["el_tau"])
    po.append(og["po_p"], og["po_tau"])
    return dict(events=(oe["n_fired"], op["n_fired"], og["n_fired"]), photons_kept=kept)
