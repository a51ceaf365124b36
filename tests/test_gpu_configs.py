"""BASELINE.json configurations on the GPU, at full size where the oracle can follow on samples.

* config 1: every element (65 536 leptons + 65 536 photons, fp64, 256 / 256x256 tables).
* config 2 (the one bench.py times), config 3, config 5 (an eighth of it; full size with PICSARQED_FULL_C5=1): the launch
  configuration of bench.py (picsarqed_qed_step on the whole population, GPU-built tables exported to the oracle),
  checked on sampled particles the oracle recomputes one by one, plus properties that hold at any size: ascending
  parent list, count = number of negative optical depths, energy conservation of every event, nothing touched
  that did not fire.
"""
import os

import numpy as np
import pytest

from parity_common import LEPTON, PHOTON, TOL_TAU, check_evolve, code, to_dev

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


def _sample_indices(n, rng, blocks=24, width=3000):
    """contiguous blocks (several compaction chunks each, tile borders included) + the first and last particles"""
    starts = rng.integers(0, max(1, n - width), size=blocks)
    starts = np.concatenate([starts, [0, max(0, n - width), (n // 2 // 4096) * 4096 - width // 2]])
    idx = np.unique(np.concatenate([np.arange(s, min(s + width, n)) for s in starts if s >= 0]))
    return idx


def _vec_ok(got, ref, tol):
    ref = [np.asarray(a, np.float64) for a in ref]
    norm = np.sqrt(sum(a * a for a in ref))
    return all(np.all(np.abs(np.asarray(g_, np.float64) - r_) <= tol * norm) for g_, r_ in zip(got, ref))


def _step_and_check(orc, qed, ctx, tabs, species, dtype, tdtype, dp, de, db, dtau, dt, seed, step, id_base, rng):
    """one qed_step on device state (dp, dtau updated in place); returns number of events"""
    import torch
    n = dtau.numel()
    tabs_r = tabs.with_fp32_reads(np.dtype(dtype) == np.float32)
    S = _sample_indices(n, rng)
    St = torch.from_numpy(S).cuda()
    p0 = [t[St].cpu().numpy() for t in dp]
    e0 = [t[St].cpu().numpy() for t in de]
    b0 = [t[St].cpu().numpy() for t in db]
    tau0 = dtau[St].cpu().numpy()
    # (a) evolve alone on a copy: sampled parity with the tie protocol; its flags define the expected count
    tau_mid = dtau.clone()
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    ctx.evolve_optical_depth(species, dp, de, db, dt, tau_mid, cnt)
    o = orc.evolve_optical_depth(tabs_r, species, code(tdtype), p0, e0, b0, dt, tau0)
    ln_chi = np.log(np.maximum(orc.chi(species, p0, e0, b0), 1e-300))
    tau_mid_s = tau_mid[St].cpu().numpy()
    n_amb, _ = check_evolve(tau_mid_s, tau0.astype(np.float64), o, dtype, ln_chi)
    assert n_amb <= 8
    fired_mask = tau_mid < 0
    n_fired = int(fired_mask.sum().item())
    assert ctx.read_count(cnt) == n_fired
    # (b) the whole step, as bench.py launches it
    cap = n_fired + 16
    nsec = 1 if species == LEPTON else 2
    sec_p = [[torch.full((cap,), -7.0, dtype=dp[0].dtype, device="cuda") for _ in range(3)] for _ in range(nsec)]
    sec_t = [torch.full((cap,), -7.0, dtype=dtau.dtype, device="cuda") for _ in range(nsec)]
    parent = torch.full((cap,), -1, dtype=torch.int64, device="cuda")
    n_out = torch.zeros(1, dtype=torch.int64, device="cuda")
    p_before = [t.clone() for t in dp]
    ctx.qed_step(species, dp, de, db, dtau, dt, seed, step, id_base, cap, sec_p[0], sec_t[0],
                 sec_p[1] if nsec == 2 else None, sec_t[1] if nsec == 2 else None, parent, n_out)
    assert ctx.read_count(n_out) == n_fired                                   # count, bit-exact
    par = parent[:n_fired]
    assert bool((par[1:] > par[:-1]).all())                                    # ascending parent index
    assert torch.equal(par, torch.nonzero(fired_mask).flatten())               # exactly the fired particles, in order
    assert bool((parent[n_fired:] == -1).all()) and bool((sec_t[0][n_fired:] == -7.0).all())
    untouched = ~fired_mask
    for a_, b_ in zip(dp, p_before):
        assert torch.equal(a_[untouched], b_[untouched])
    assert torch.equal(dtau[untouched], tau_mid[untouched])
    # energy bookkeeping of every event, in fp64 on the device
    pb = [t[par].double() for t in p_before]
    pa = [t[par].double() for t in dp]
    norm = lambda v: torch.sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2])
    tol = TOL_TAU[np.dtype(dtype)]
    if species == LEPTON:
        g_b, g_a = torch.sqrt(1 + norm(pb) ** 2), torch.sqrt(1 + norm(pa) ** 2)
        g_ph = norm([t[:n_fired].double() for t in sec_p[0]])
        assert bool((torch.abs(g_b - g_a - g_ph) <= 4 * tol * g_b).all())     # gamma' + gamma_gamma = gamma
        assert bool((g_ph < g_b - 1).all()) and bool((dtau[par] > 0).all())
    else:
        gg = norm(pb)
        g_e = torch.sqrt(1 + norm([t[:n_fired].double() for t in sec_p[0]]) ** 2)
        g_p = torch.sqrt(1 + norm([t[:n_fired].double() for t in sec_p[1]]) ** 2)
        assert bool((torch.abs(g_e + g_p - gg) <= 4 * tol * gg).all())         # gamma_- + gamma_+ = gamma_gamma
        assert bool((norm(pa) == 0).all()) and bool(torch.isinf(dtau[par]).all())
    # (c) sampled events against the oracle (the oracle gets the GPU's evolved tau of the sample)
    ids = (id_base + S).astype(np.uint64)
    if species == LEPTON:
        oe = orc.generate_photons(tabs_r, code(dtype), code(tdtype), p0, e0, b0, tau_mid_s, seed, step, ids)
        o_sec, o_sect = [oe["ph_p"]], [oe["ph_tau"]]
    else:
        oe = orc.generate_pairs(tabs_r, code(dtype), code(tdtype), p0, e0, b0, tau_mid_s, seed, step, ids)
        o_sec, o_sect = [oe["el_p"], oe["po_p"]], [oe["el_tau"], oe["po_tau"]]
    fired_global = S[oe["parent"]]
    slots = torch.searchsorted(par, torch.from_numpy(fired_global).cuda())
    assert torch.equal(par[slots], torch.from_numpy(fired_global).cuda())
    ttol = TOL_TAU[np.dtype(tdtype)]
    for s in range(nsec):
        assert _vec_ok([t[slots].cpu().numpy() for t in sec_p[s]], o_sec[s], tol)
        got_t = sec_t[s][slots].cpu().numpy().astype(np.float64)
        assert np.all(np.abs(got_t - o_sect[s]) <= ttol * o_sect[s])
    p_after_s = [t[St].cpu().numpy() for t in dp]
    if species == LEPTON:
        assert _vec_ok(p_after_s, oe["p"], tol)
    tau_after_s = dtau[St].cpu().numpy().astype(np.float64)
    fin = np.isfinite(oe["tau"])
    assert np.array_equal(np.isfinite(tau_after_s), fin)
    assert np.all(np.abs(tau_after_s[fin] - oe["tau"][fin]) <= ttol * np.abs(oe["tau"][fin]))
    return n_fired


def _dt_from_gpu(qed, ctx, species, dp, de, db, m=65536):
    import torch
    probe = torch.zeros(m, dtype=torch.float64 if dp[0].dtype == torch.float64 else torch.float32, device="cuda")
    ctx.evolve_optical_depth(species, [t[:m] for t in dp], [t[:m] for t in de], [t[:m] for t in db], 1.0, probe)
    return qed.workloads.choose_dt((-probe).double().cpu().numpy(), 0.05)


def test_config1_every_element(orc, qed):
    """BASELINE config 1: tiny mixed step, fp64, all elements against the oracle"""
    import torch
    ctx, tabs = _ctx_with_tables(orc, qed, 1)
    n, seed = 65536, 1
    pops = {sp: qed.workloads.config1(seed=seed, n=n, species=sp) for sp in (LEPTON, PHOTON)}
    rates = np.concatenate([orc.rate(tabs, sp, *pops[sp])[:32768] for sp in (LEPTON, PHOTON)])
    dt = qed.workloads.choose_dt(rates, 0.05)        # ~5 % of the particles fire, over both species
    fired_total = 0
    for sp in (LEPTON, PHOTON):
        p, e, b = pops[sp]
        dp, de, db = to_dev(p), to_dev(e), to_dev(b)
        tau = torch.empty(n, dtype=torch.float64, device="cuda")
        ctx.init_optical_depth(sp, tau, seed, sp * n)
        tau0 = tau.cpu().numpy()
        assert np.allclose(tau0, orc.init_optical_depth(sp, 1, n, seed, ids=sp * n + np.arange(n, dtype=np.uint64)),
                           rtol=1e-14, atol=0)
        nsec = 1 if sp == LEPTON else 2
        sec_p = [[torch.zeros(n, dtype=torch.float64, device="cuda") for _ in range(3)] for _ in range(nsec)]
        sec_t = [torch.zeros(n, dtype=torch.float64, device="cuda") for _ in range(nsec)]
        parent = torch.zeros(n, dtype=torch.int64, device="cuda")
        n_out = torch.zeros(1, dtype=torch.int64, device="cuda")
        # the evolve pass of the step, seen through picsarqed_evolve_optical_depth on a copy (the same kernel arithmetic;
        # tests/test_gpu_parity.py::test_fused_step holds the two bit-identical): the GPU's evolved tau of EVERY particle
        tau_mid_d = tau.clone()
        ctx.evolve_optical_depth(sp, dp, de, db, dt, tau_mid_d)
        tau_mid = tau_mid_d.cpu().numpy()
        ctx.qed_step(sp, dp, de, db, tau, dt, seed, 0, sp * n, n, sec_p[0], sec_t[0], sec_p[1] if nsec == 2 else None,
                     sec_t[1] if nsec == 2 else None, parent, n_out)
        k = ctx.read_count(n_out)
        o = orc.evolve_optical_depth(tabs, sp, 1, p, e, b, dt, tau0)
        ln_chi = np.log(np.maximum(orc.chi(sp, p, e, b), 1e-300))
        fired = np.zeros(n, bool)
        fired[parent.cpu().numpy()[:k]] = True
        n_amb, flags = check_evolve(tau_mid, tau0, o, np.float64, ln_chi)
        assert n_amb == 0 and np.array_equal(flags, fired) and k == int((o["tau"] < 0).sum())
        assert np.array_equal(tau.cpu().numpy()[~fired], tau_mid[~fired])   # the step left the others as the evolve pass did
        ids = sp * n + np.arange(n, dtype=np.uint64)
        if sp == LEPTON:
            oe = orc.generate_photons(tabs, 1, 1, p, e, b, o["tau"], seed, 0, ids)
            o_sec, o_sect = [oe["ph_p"]], [oe["ph_tau"]]
        else:
            oe = orc.generate_pairs(tabs, 1, 1, p, e, b, o["tau"], seed, 0, ids)
            o_sec, o_sect = [oe["el_p"], oe["po_p"]], [oe["el_tau"], oe["po_tau"]]
        assert np.array_equal(parent.cpu().numpy()[:k], oe["parent"])          # compaction order, bit-exact
        for s in range(nsec):
            assert _vec_ok([t.cpu().numpy()[:k] for t in sec_p[s]], o_sec[s], 1e-9)
            assert np.allclose(sec_t[s].cpu().numpy()[:k], o_sect[s], rtol=1e-9, atol=0)
        assert _vec_ok([t.cpu().numpy() for t in dp], oe["p"], 1e-9) or sp == PHOTON
        fin = np.isfinite(oe["tau"])
        got = tau.cpu().numpy()
        assert np.array_equal(np.isfinite(got), fin)
        assert np.all(np.abs(got[fin] - oe["tau"][fin]) <= 1e-9 * (np.abs(oe["tau"][fin]) + o["decr"][fin]))
        fired_total += k
    assert 0.03 < fired_total / (2 * n) < 0.07
    ctx.close()


def test_config2_bench_configuration(orc, qed):
    """BASELINE config 2 as bench.py runs it: 16 Mi electrons, fp64, 1024 / 1024x1024 tables, fields re-drawn per step"""
    import torch
    ctx, tabs = _ctx_with_tables(orc, qed, 2)
    n, seed = 1 << 24, 2
    p_h, gamma = qed.workloads.config2(seed=seed, n=n)
    dp = to_dev(p_h)
    tau = torch.empty(n, dtype=torch.float64, device="cuda")
    ctx.init_optical_depth(LEPTON, tau, seed, 0)
    rng = np.random.default_rng(20)
    dt = None
    for step in range(2):
        e_h, b_h = qed.workloads.config2_fields(seed, step, gamma)
        de, db = to_dev(e_h), to_dev(b_h)
        if dt is None:
            dt = _dt_from_gpu(qed, ctx, LEPTON, dp, de, db)
        k = _step_and_check(orc, qed, ctx, tabs, LEPTON, np.float64, np.float64, dp, de, db, tau, dt, seed, step, 0, rng)
        assert 0.02 < k / n < 0.1
    ctx.close()


def test_config3_pair_production_fp32(orc, qed):
    """BASELINE config 3: 16 Mi photons, fp32, BW table 1024 / 1024x1024 read through its fp32 copy"""
    import torch
    ctx, tabs = _ctx_with_tables(orc, qed, 3)
    n, seed = 1 << 24, 3
    p_h, gamma = qed.workloads.config3(seed=seed, n=n)
    dp = to_dev(p_h)
    tau = torch.empty(n, dtype=torch.float32, device="cuda")
    ctx.init_optical_depth(PHOTON, tau, seed, 0)
    rng = np.random.default_rng(30)
    e_h, b_h = qed.workloads.config3_fields(seed, 0, gamma)
    de, db = to_dev(e_h), to_dev(b_h)
    dt = _dt_from_gpu(qed, ctx, PHOTON, dp, de, db)
    k = _step_and_check(orc, qed, ctx, tabs, PHOTON, np.float32, np.float32, dp, de, db, tau, dt, seed, 0, 0, rng)
    assert 0.02 < k / n < 0.1
    ctx.close()


def test_config5_mixed_precision(orc, qed):
    """BASELINE config 5: fp32 particles with fp64 optical depth, laser-plasma-like fields, both species.
    An eighth of the size by default (the 10-step test of tests/test_gpu_config_length.py runs 256 Mi + 64 Mi);
    PICSARQED_FULL_C5=1 runs the full size here as well."""
    import torch
    full = os.environ.get("PICSARQED_FULL_C5") == "1"   # (tests/test_gpu_config_length.py runs the full size, 10 steps)
    n_lep, n_pho = ((1 << 28), (1 << 26)) if full else ((1 << 25), (1 << 23))
    ctx, tabs = _ctx_with_tables(orc, qed, 5)
    rng = np.random.default_rng(50)
    id_base = 0
    for sp, n in ((LEPTON, n_lep), (PHOTON, n_pho)):
        p, e, b = qed.workloads.config5(seed=5, n=n, species=sp)
        dp, de, db = to_dev(p), to_dev(e), to_dev(b)
        del p, e, b
        tau = torch.empty(n, dtype=torch.float64, device="cuda")
        ctx.init_optical_depth(sp, tau, 5, id_base)
        dt = _dt_from_gpu(qed, ctx, sp, dp, de, db)
        k = _step_and_check(orc, qed, ctx, tabs, sp, np.float32, np.float64, dp, de, db, tau, dt, 5, 0, id_base, rng)
        assert 0.005 < k / n < 0.12
        id_base += n
        del dp, de, db, tau
        torch.cuda.empty_cache()
    ctx.close()
