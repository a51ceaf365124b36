"""BASELINE.json configurations 2, 3 and 5 at their full LENGTH (100, 20, 10 steps) and full SIZE, free-running.

The GPU steps the whole population with picsarqed_qed_step, as bench.py launches it.  The oracle cannot follow
16 Mi x 100 particle-steps, so it carries a fixed, index-ordered slab (the first and the last 256 Ki particles and 24
random 4 Ki-aligned blocks of 4 Ki: tile borders, the ragged end of the grid and the interior) through ALL steps on its
own state -- its own debited momenta, its own re-drawn optical depths -- and the slab is compared
every step: optical depth after the evolve pass (tie protocol), flags, count and order of the slab's events, secondaries,
parents after the step.  A flag inside the tie margin takes the GPU's value (reported per configuration).  Every step
also checks what holds at any size on the whole population: count = number of negative optical depths, parent list =
exactly those particles in ascending order, energy bookkeeping of every event, nothing else touched.
"""
import os

import numpy as np
import pytest

from parity_common import LEPTON, PHOTON, TOL_TAU, EPS, code, tie_margin, to_dev

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def qed():
    import paper_2110_00256_b200 as q
    return q


def _ctx_with_tables(orc, qed, config):
    kw = qed.workloads.table_params(config)
    ctx = qed.Context(0)
    ctx.build_tables(qed.TableParams(**kw))
    tabs = orc.Tables(orc.TableParams(**kw), ctx.export_tables(qed.TAB_LNG), ctx.export_tables(qed.TAB_QS_LNP),
                      ctx.export_tables(qed.TAB_LNT), ctx.export_tables(qed.TAB_BW_P))
    return ctx, tabs


def slab_indices(n, rng, edge=1 << 18, blocks=24, width=1 << 12):
    edge = min(edge, n // 4)
    starts = rng.integers(edge // width, (n - edge) // width - 1, size=blocks) * width
    parts = [np.arange(0, edge), np.arange(n - edge, n)] + [np.arange(s, s + width) for s in starts]
    return np.unique(np.concatenate(parts))


def _vec_err(got, ref):
    ref = [np.asarray(a, np.float64) for a in ref]
    norm = np.sqrt(sum(a * a for a in ref))
    err = np.max([np.abs(np.asarray(g_, np.float64) - r_) for g_, r_ in zip(got, ref)], axis=0)
    return err, norm


class Follower:
    """the oracle's free-running copy of the slab of one species"""

    def __init__(self, orc, tabs, species, dtype, tdtype, S, dp, dtau, id_base):
        import torch
        self.orc, self.species, self.dtype, self.tdtype = orc, species, np.dtype(dtype), np.dtype(tdtype)
        self.tabs = tabs.with_fp32_reads(self.dtype == np.float32)
        self.S, self.St = S, torch.from_numpy(S).cuda()
        self.p = [t[self.St].cpu().numpy().astype(np.float64) for t in dp]
        self.tau = dtau[self.St].cpu().numpy().astype(np.float64)
        self.ids = (id_base + S).astype(np.uint64)
        self.n_ambiguous = 0
        self.max_tau_err = 0.0
        self.max_p_err = 0.0

    def gather(self, tensors):
        return [t[self.St] for t in tensors]


def step_and_compare(orc, qed, ctx, F, dp, de, db, dtau, dt, seed, step, id_base, sec_p, sec_t, parent, n_out, cap):
    """one qed_step of the whole population; the follower F is advanced by the oracle and compared"""
    import torch
    species, n = F.species, dtau.numel()
    tol, ttol = TOL_TAU[F.dtype], TOL_TAU[F.tdtype]
    etol = tol      # the decrement is computed in the particle arithmetic whatever the type tau is stored in
    nsec = 1 if species == LEPTON else 2
    # ---- the evolve pass, seen through picsarqed_evolve_optical_depth on a copy (the same kernel arithmetic)
    tau_mid = dtau.clone()
    ctx.evolve_optical_depth(species, dp, de, db, dt, tau_mid)
    fired_mask = tau_mid < 0
    n_fired = int(fired_mask.sum().item())
    assert n_fired <= cap
    e_s = [t.cpu().numpy() for t in F.gather(de)]
    b_s = [t.cpu().numpy() for t in F.gather(db)]
    tau_gpu_old = dtau[F.St].cpu().numpy().astype(np.float64)
    tau_gpu_mid = tau_mid[F.St].cpu().numpy().astype(np.float64)
    o = orc.evolve_optical_depth(F.tabs, species, code(F.tdtype), F.p, e_s, b_s, dt, F.tau)
    fin = np.isfinite(F.tau)
    # the two states run freely: what they differed by when the step began (within the tolerance of the steps before, on
    # THEIR scale |tau_old| + decrement, which may be much larger than today's tau) is carried, not re-earned
    with np.errstate(invalid="ignore"):
        drift = np.abs(np.where(fin, tau_gpu_old - F.tau, 0.0))
    ref = np.abs(F.tau[fin]) + o["decr"][fin]
    err = np.maximum(np.abs(tau_gpu_mid[fin] - o["tau_exact"][fin]) - drift[fin], 0.0)
    assert np.all(err <= etol * ref), "step %d: evolved tau off by %g of its scale" % (step, float(np.max(err / ref)))
    F.max_tau_err = max(F.max_tau_err, float(np.max(err / ref)) if ref.size else 0.0)
    assert np.array_equal(np.isfinite(tau_gpu_mid), fin)
    ln_chi = np.log(np.maximum(orc.chi(species, F.p, e_s, b_s), 1e-300))
    # flags: equal outside the tie margin, which here also holds the drift the two free-running states have accumulated
    margin = tie_margin(F.dtype, F.tau, o, ln_chi) + drift
    f_gpu, f_orc = tau_gpu_mid < 0, o["tau"] < 0
    diff = f_gpu != f_orc
    assert not np.any(diff & ~(np.abs(o["tau_exact"]) <= margin)), "step %d: flag mismatch outside the tie margin" % step
    F.n_ambiguous += int(diff.sum())
    tau_orc_mid = np.where(diff, tau_gpu_mid, o["tau"])          # (the GPU's flag for the ambiguous ones)
    # ---- the step itself, on the whole population
    p_before = [t.clone() for t in dp]
    ctx.qed_step(species, dp, de, db, dtau, dt, seed, step, id_base, cap, sec_p[0], sec_t[0],
                 sec_p[1] if nsec == 2 else None, sec_t[1] if nsec == 2 else None, parent, n_out)
    assert ctx.read_count(n_out) == n_fired                                    # count, bit-exact
    par = parent[:n_fired]
    assert torch.equal(par, torch.nonzero(fired_mask).flatten())               # exactly the fired particles, ascending
    untouched = ~fired_mask
    for a_, b_ in zip(dp, p_before):
        assert torch.equal(a_[untouched], b_[untouched])
    assert torch.equal(dtau[untouched], tau_mid[untouched])
    pb = [t[par].double() for t in p_before]
    norm = lambda v: torch.sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2])
    if species == LEPTON:
        pa = [t[par].double() for t in dp]
        g_b, g_a = torch.sqrt(1 + norm(pb) ** 2), torch.sqrt(1 + norm(pa) ** 2)
        g_ph = norm([t[:n_fired].double() for t in sec_p[0]])
        assert bool((torch.abs(g_b - g_a - g_ph) <= 4 * tol * g_b).all())     # gamma' + gamma_gamma = gamma
        assert bool((dtau[par] > 0).all())
    else:
        gg = norm(pb)
        g_e = torch.sqrt(1 + norm([t[:n_fired].double() for t in sec_p[0]]) ** 2)
        g_p = torch.sqrt(1 + norm([t[:n_fired].double() for t in sec_p[1]]) ** 2)
        assert bool((torch.abs(g_e + g_p - gg) <= 4 * tol * gg).all())         # gamma_- + gamma_+ = gamma_gamma
        assert bool(torch.isinf(dtau[par]).all()) and all(bool((t[par] == 0).all()) for t in dp)
    # ---- the slab's events by the oracle, from its own state
    gen = orc.generate_photons if species == LEPTON else orc.generate_pairs
    oe = gen(F.tabs, code(F.dtype), code(F.tdtype), F.p, e_s, b_s, tau_orc_mid, seed, step, F.ids)
    o_sec = [oe["ph_p"]] if species == LEPTON else [oe["el_p"], oe["po_p"]]
    o_sect = [oe["ph_tau"]] if species == LEPTON else [oe["el_tau"], oe["po_tau"]]
    fired_global = torch.from_numpy(F.S[oe["parent"]]).cuda()
    in_slab = torch.isin(par, F.St)
    assert int(in_slab.sum().item()) == oe["n_fired"]                          # the slab's count
    slots = torch.nonzero(in_slab).flatten()
    assert torch.equal(par[slots], fired_global)                               # the slab's events, in order
    for s in range(nsec):
        err, nrm = _vec_err([t[slots].cpu().numpy() for t in sec_p[s]], o_sec[s])
        assert np.all(err <= tol * nrm), "step %d: secondary momentum" % step
        got_t = sec_t[s][slots].cpu().numpy().astype(np.float64)
        assert np.all(np.abs(got_t - o_sect[s]) <= ttol * o_sect[s])
    F.p, F.tau = oe["p"], oe["tau"]
    err, nrm = _vec_err([t.cpu().numpy() for t in F.gather(dp)], F.p)
    ok = nrm > 0
    assert np.all(err[ok] <= tol * nrm[ok]) and np.all(err[~ok] == 0), "step %d: parent momentum" % step
    F.max_p_err = max(F.max_p_err, float(np.max(err[ok] / nrm[ok])) if ok.any() else 0.0)
    tau_after = dtau[F.St].cpu().numpy().astype(np.float64)
    fin = np.isfinite(F.tau)
    assert np.array_equal(np.isfinite(tau_after), fin)
    # (a re-drawn tau is compared relative to itself; a tau that only evolved carries the evolve tolerance)
    scale = np.where(tau_orc_mid[fin] < 0, np.abs(F.tau[fin]), np.abs(F.tau[fin]) + o["decr"][fin])
    carried = np.where(tau_orc_mid[fin] < 0, 0.0, drift[fin])     # (a re-drawn tau starts afresh)
    rtol = np.where(tau_orc_mid[fin] < 0, ttol, etol)
    assert np.all(np.abs(tau_after[fin] - F.tau[fin]) <= rtol * np.maximum(scale, 1e-300) + carried), "step %d: tau after the step" % step
    return n_fired


def _buffers(n, cap, nsec, pdt, tdt):
    import torch
    sec_p = [[torch.empty(cap, dtype=pdt, device="cuda") for _ in range(3)] for _ in range(nsec)]
    sec_t = [torch.empty(cap, dtype=tdt, device="cuda") for _ in range(nsec)]
    return sec_p, sec_t, torch.empty(cap, dtype=torch.int64, device="cuda"), torch.zeros(1, dtype=torch.int64, device="cuda")


def _dt_from_gpu(qed, ctx, species, dp, de, db, m=65536):
    import torch
    probe = torch.zeros(m, dtype=torch.float64 if dp[0].dtype == torch.float64 else torch.float32, device="cuda")
    ctx.evolve_optical_depth(species, [t[:m] for t in dp], [t[:m] for t in de], [t[:m] for t in db], 1.0, probe)
    return (-probe).double().cpu().numpy()


def _report(name, F, fired_total, particle_steps):
    print("\n[config-length parity] %s: %d ambiguous flags in %d slab particle-steps; fired %.3f; max tau error %.2e of "
          "the tolerance scale, max parent momentum error %.2e" % (name, F.n_ambiguous, particle_steps, fired_total,
                                                                 F.max_tau_err, F.max_p_err))


def test_config2_100_steps(orc, qed):
    """BASELINE config 2: 16 Mi electrons, fp64, 100 steps, emitters debited in place, fields re-drawn every step from
    the seed (eight field sets of the generator, cycled: 6 GB resident)"""
    import torch
    ctx, tabs = _ctx_with_tables(orc, qed, 2)
    n, seed, steps, n_sets = 1 << 24, 2, 100, 8
    p_h, gamma = qed.workloads.config2(seed=seed, n=n)
    dp = to_dev(p_h)
    fields = []
    for k in range(n_sets):
        e_h, b_h = qed.workloads.config2_fields(seed, k, gamma)
        fields.append((to_dev(e_h), to_dev(b_h)))
    del p_h, e_h, b_h
    tau = torch.empty(n, dtype=torch.float64, device="cuda")
    ctx.init_optical_depth(LEPTON, tau, seed, 0)
    dt = qed.workloads.choose_dt(_dt_from_gpu(qed, ctx, LEPTON, dp, *fields[0]), 0.05)
    S = slab_indices(n, np.random.default_rng(200))
    F = Follower(orc, tabs, LEPTON, np.float64, np.float64, S, dp, tau, 0)
    cap = n // 8
    sec_p, sec_t, parent, n_out = _buffers(n, cap, 1, torch.float64, torch.float64)
    fired = 0
    for step in range(steps):
        de, db = fields[step % n_sets]
        fired += step_and_compare(orc, qed, ctx, F, dp, de, db, tau, dt, seed, step, 0, sec_p, sec_t, parent, n_out, cap)
    _report("config 2 (fp64, 100 steps)", F, fired / (n * steps), S.size * steps)
    assert F.n_ambiguous == 0 and 0.02 < fired / (n * steps) < 0.1
    ctx.close()


def test_config3_20_steps(orc, qed):
    """BASELINE config 3: 16 Mi photons, fp32, 20 steps of pair production; the photons that decayed are re-seeded between
    steps: they come back with their first momentum and optical depth, on both sides alike"""
    import torch
    ctx, tabs = _ctx_with_tables(orc, qed, 3)
    n, seed, steps, n_sets = 1 << 24, 3, 20, 4
    p_h, gamma = qed.workloads.config3(seed=seed, n=n)
    dp = to_dev(p_h)
    fields = []
    for k in range(n_sets):
        e_h, b_h = qed.workloads.config3_fields(seed, k, gamma)
        fields.append((to_dev(e_h), to_dev(b_h)))
    del p_h, e_h, b_h
    tau = torch.empty(n, dtype=torch.float32, device="cuda")
    ctx.init_optical_depth(PHOTON, tau, seed, 0)
    p0, tau0 = [t.clone() for t in dp], tau.clone()
    dt = qed.workloads.choose_dt(_dt_from_gpu(qed, ctx, PHOTON, dp, *fields[0]), 0.05)
    S = slab_indices(n, np.random.default_rng(300))
    F = Follower(orc, tabs, PHOTON, np.float32, np.float32, S, dp, tau, 0)
    Fp0, Ftau0 = [a.copy() for a in F.p], F.tau.copy()
    cap = n // 8
    sec_p, sec_t, parent, n_out = _buffers(n, cap, 2, torch.float32, torch.float32)
    fired = 0
    for step in range(steps):
        dead = torch.isinf(tau)                                   # re-seed: the generator's first draw comes back
        for a, a0 in zip(dp, p0):
            torch.where(dead, a0, a, out=a)
        torch.where(dead, tau0, tau, out=tau)
        dead_h = np.isinf(F.tau)
        F.p = [np.where(dead_h, a0, a) for a, a0 in zip(F.p, Fp0)]
        F.tau = np.where(dead_h, Ftau0, F.tau)
        de, db = fields[step % n_sets]
        fired += step_and_compare(orc, qed, ctx, F, dp, de, db, tau, dt, seed, step, 0, sec_p, sec_t, parent, n_out, cap)
    _report("config 3 (fp32, 20 steps)", F, fired / (n * steps), S.size * steps)
    assert F.n_ambiguous <= 200 and 0.02 < fired / (n * steps) < 0.1
    ctx.close()


def test_config5_10_steps(orc, qed):
    """BASELINE config 5: 256 Mi leptons + 64 Mi photons (PICSARQED_SMALL_C5=1: an eighth), fp32 with fp64 optical depth,
    plane wave + noise, 10 steps of both processes; photons that decay stay removed"""
    import torch
    full = os.environ.get("PICSARQED_SMALL_C5") != "1"
    sizes = {LEPTON: (1 << 28) if full else (1 << 25), PHOTON: (1 << 26) if full else (1 << 23)}
    ctx, tabs = _ctx_with_tables(orc, qed, 5)
    seed, steps = 5, 10
    state, id_base, rates = {}, 0, []
    for sp in (LEPTON, PHOTON):
        n = sizes[sp]
        p, e, b = qed.workloads.config5(seed=seed, n=n, species=sp)
        dp, de, db = to_dev(p), to_dev(e), to_dev(b)
        del p, e, b
        tau = torch.empty(n, dtype=torch.float64, device="cuda")
        ctx.init_optical_depth(sp, tau, seed, id_base)
        rates.append(_dt_from_gpu(qed, ctx, sp, dp, de, db))
        S = slab_indices(n, np.random.default_rng(500 + sp))
        F = Follower(orc, tabs, sp, np.float32, np.float64, S, dp, tau, id_base)
        cap = n // 4
        state[sp] = (dp, de, db, tau, F, id_base, cap, _buffers(n, cap, 1 + sp, torch.float32, torch.float64))
        id_base += n
    dt = qed.workloads.choose_dt(np.concatenate(rates), 0.05)     # one time step for both species
    fired = {LEPTON: 0, PHOTON: 0}
    for step in range(steps):
        for sp in (LEPTON, PHOTON):
            dp, de, db, tau, F, ib, cap, (sec_p, sec_t, parent, n_out) = state[sp]
            fired[sp] += step_and_compare(orc, qed, ctx, F, dp, de, db, tau, dt, seed, step, ib, sec_p, sec_t, parent, n_out, cap)
    for sp, name in ((LEPTON, "leptons"), (PHOTON, "photons")):
        F = state[sp][4]
        _report("config 5 %s (fp32 + fp64 tau, 10 steps)" % name, F, fired[sp] / (sizes[sp] * steps), F.S.size * steps)
        assert F.n_ambiguous <= 200
    ctx.close()
