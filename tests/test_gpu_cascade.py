"""GPU parity of the closed loop in a uniform field: Boris push, ordered filtering
append, energy spectrum and the whole cascade step, through the C ABI, against oracle/cascade.py on the same seeded
inputs and table bytes."""
import numpy as np
import pytest

from parity_common import LEPTON, PHOTON, code, to_dev, to_host

pytestmark = pytest.mark.gpu

ID_BASE = {"electrons": 0, "positrons": 1 << 40, "photons": 1 << 41}   # DESIGN.md R21 (typed here, not imported)


@pytest.fixture(scope="module")
def qed():
    import paper_2110_00256_b200 as q
    return q


@pytest.fixture(scope="module")
def cas():
    from oracle import cascade
    return cascade


@pytest.fixture(scope="module")
def mid_tables(orc):
    p = orc.TableParams(qs_chi_min=1e-3, qs_chi_max=1e3, qs_n_chi=40, qs_xi_min=1e-12, qs_n_xi=96,
                        bw_chi_min=2e-2, bw_chi_max=1e3, bw_n_chi=40, bw_n_xi=96)
    return orc.build_tables(p)


@pytest.fixture(scope="module")
def ctx(qed, mid_tables):
    c = qed.Context(0)
    tp = mid_tables.params
    c.import_tables(qed.TableParams(**{k: getattr(tp, k) for k in tp.__dataclass_fields__}), mid_tables.lnG,
                    mid_tables.qs_lnP, mid_tables.lnT, mid_tables.bw_P)
    yield c
    c.close()


def _momenta(n, seed, dtype, lo=1e-2, hi=1e4):
    """isotropic directions, magnitude log-uniform on [lo, hi]"""
    rng = np.random.default_rng(seed)
    d = rng.standard_normal((3, n))
    d /= np.linalg.norm(d, axis=0)
    mag = np.exp(rng.uniform(np.log(lo), np.log(hi), n))
    return [np.ascontiguousarray((d[c] * mag).astype(dtype)) for c in range(3)]


# ----------------------------------------------------------------------------- Boris push
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("n", [100003, 6, 1])
def test_boris_push(qed, ctx, cas, dtype, n):
    """per component, relative to |u|: 1e-12 (fp64: the kernel's 1/sqrt and 1/x are few-ulp) / 2e-7 (fp32: the
    arithmetic is fp64, the result is rounded once to fp32)"""
    p = _momenta(n, 3, dtype)
    tol = 1e-12 if dtype == np.float64 else 2e-7
    for sign, e, b, dt in ((-1, (0, 0, 0), (0, 0, 1e-3), 2e-18), (+1, (2e-4, -1e-4, 3e-5), (1e-3, 5e-4, -2e-3), 1e-18),
                           (-1, (1e-3, 0, 0), (0, 0, 0), 5e-19), (+1, (0, 0, 0), (0, 9e-3, 0), 4e-17)):
        ref = cas.boris_push_uniform(p, sign, e, b, dt)
        dp = to_dev(p)
        ctx.boris_push_uniform(dp, sign, e, b, dt)
        got = to_host(dp)
        norm = np.sqrt(sum(a.astype(np.float64) ** 2 for a in ref))
        for c in range(3):
            assert np.all(np.abs(got[c].astype(np.float64) - ref[c]) <= tol * norm + 1e-300), (sign, e, b, c)
        if e == (0, 0, 0) and dtype == np.float64:   # pure rotation keeps |u|
            assert np.allclose(np.sqrt(sum(a * a for a in got)), np.sqrt(sum(a * a for a in p)), rtol=1e-14)


# ----------------------------------------------------------------------------- ordered filtering append
@pytest.mark.parametrize("dtype,tdtype", [(np.float64, np.float64), (np.float32, np.float32), (np.float32, np.float64)])
@pytest.mark.parametrize("m_max,count", [(100003, 100003), (100003, 77001), (4096, 5000), (128, 128), (5, 3), (7, 0)])
def test_append_secondaries(qed, ctx, cas, dtype, tdtype, m_max, count):
    """bit-exact: which entries are kept (strict < threshold in fp64, R22), their order, where they land, the new
    count; entries past the destination's capacity are not written"""
    import torch
    src = _momenta(m_max, 4, dtype, lo=1e-2, hi=1e2)
    rng = np.random.default_rng(44)
    stau = rng.exponential(size=m_max).astype(tdtype)
    m = min(m_max, count)
    dst_n = 37
    for thr in (0.0, 2.0, 1e9):
        g = np.sqrt(src[0].astype(np.float64) ** 2 + src[1].astype(np.float64) ** 2 + src[2].astype(np.float64) ** 2)
        keep = cas.keep_photons([a[:m].astype(np.float64) for a in src], thr)
        assert np.array_equal(keep, ~(g[:m] < thr))
        kept = int(keep.sum())
        for cap in (dst_n + m_max, dst_n + kept // 2):
            dst = [torch.full((cap,), -7.0, dtype=torch.from_numpy(src[0]).dtype, device="cuda") for _ in range(3)]
            dtau = torch.full((cap,), -7.0, dtype=torch.from_numpy(stau).dtype, device="cuda")
            cnt = torch.tensor([count], dtype=torch.int64, device="cuda")
            new_n = torch.zeros(1, dtype=torch.int64, device="cuda")
            ctx.append_secondaries(m_max, to_dev(src), torch.from_numpy(stau).cuda(), cnt, thr, dst, dtau, dst_n, new_n)
            assert int(new_n.item()) == dst_n + kept
            w = min(kept, cap - dst_n)
            for c in range(3):
                h = dst[c].cpu().numpy()
                assert np.array_equal(h[dst_n:dst_n + w], src[c][:m][keep][:w])
                assert np.all(h[:dst_n] == -7.0) and np.all(h[dst_n + w:] == -7.0)
            h = dtau.cpu().numpy()
            assert np.array_equal(h[dst_n:dst_n + w], stau[:m][keep][:w]) and np.all(h[dst_n + w:] == -7.0)


# ----------------------------------------------------------------------------- energy spectrum
@pytest.mark.parametrize("species", [LEPTON, PHOTON])
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_energy_spectrum(qed, ctx, cas, species, dtype):
    """bit-exact counts; a particle whose position in bin units is within 1e-9 of an edge may fall on either side
    (both sides take floor of an fp64 log, the two log routines differ by an ulp)"""
    import torch
    n = 300007
    p = _momenta(n, 5, dtype, lo=1e-4, hi=1e5)
    for k in range(0, n, 1000):   # dead entries
        p[0][k] = p[1][k] = p[2][k] = 0
    for lo, hi, nb in ((1e-2, 1e4, 64), (1e-3, 1e3, 8192), (1.0, 2.0, 1)):
        ref, x = cas.energy_spectrum(species, p, lo, hi, nb)
        hist = torch.zeros(nb, dtype=torch.int64, device="cuda")
        ctx.energy_spectrum(species, to_dev(p), lo, hi, hist)
        got = hist.cpu().numpy()
        xs = x[~np.isnan(x)]
        near = np.abs(xs - np.round(xs)) < 1e-9
        if not near.any():
            assert np.array_equal(got, ref)
        else:
            assert np.abs(got - ref).sum() <= 2 * near.sum() and abs(int(got.sum()) - int(ref.sum())) <= near.sum()
        assert ref.sum() > 0
        ctx.energy_spectrum(species, to_dev(p), lo, hi, hist)   # accumulates
        assert np.abs(hist.cpu().numpy() - 2 * ref).sum() <= 4 * near.sum()


# ----------------------------------------------------------------------------- the closed loop
def _start(qed, ctx, orc, cas, n, g0, seed, dtype, tdtype, cap):
    import torch
    tdt = torch.float64 if tdtype == np.float64 else torch.float32
    pdt = torch.float64 if dtype == np.float64 else torch.float32
    pops = {k: qed.Species(cap, pdt, tdt, ID_BASE[k]) for k in ("electrons", "positrons", "photons")}
    p0 = np.sqrt(g0 * g0 - 1)
    el = pops["electrons"]
    el.p[0][:n] = float(np.asarray(p0, dtype=dtype))
    el.n = n
    ctx.init_optical_depth(LEPTON, el.tau[:n], seed, ID_BASE["electrons"])
    # both sides start from the same optical depths (the GPU's -ln U is within an ulp or two of the oracle's:
    # test_gpu_parity.py::test_init_optical_depth; here the common start makes the free run comparable)
    tau0 = el.tau[:n].cpu().numpy().astype(np.float64)
    ref = orc.init_optical_depth(LEPTON, code(tdtype), n, seed, np.arange(n, dtype=np.uint64))
    assert np.allclose(tau0, ref, rtol=1e-6 if tdtype == np.float32 else 1e-14, atol=1e-15)
    o_el = cas.Population([np.full(n, float(np.asarray(p0, dtype=dtype))), np.zeros(n), np.zeros(n)], tau0)
    return pops, {"electrons": o_el, "positrons": cas.empty_population(), "photons": cas.empty_population()}


def _state(pop):
    n = pop.n
    return [t[:n].cpu().numpy().astype(np.float64) for t in pop.p], pop.tau[:n].cpu().numpy().astype(np.float64)


@pytest.mark.parametrize("b0,steps,total_time,thr", [(9e-3, 40, 1e-16, 0.0), (9e-3, 40, 1e-16, 2.0), (1e-3, 25, 1e-15, 2.0)])
def test_cascade_free_running_fp64(orc, qed, ctx, cas, mid_tables, b0, steps, total_time, thr):
    """Ridgers cases (iii) and (i), free running on both sides from the same start: after every
    step the three populations have the same sizes and the same event counts; at the end every particle agrees to
    1e-9 (relative to its momentum) and dead photons coincide.  (fp64 flags have no observed ties; a single one would
    show up as a count mismatch.)"""
    n, g0 = 4000, 1000.0
    pops, opops = _start(qed, ctx, orc, cas, n, g0, 21, np.float64, np.float64, 40 * n)
    e, b = (0.0, 0.0, 0.0), (0.0, 0.0, b0)
    dt = total_time / steps
    tot = np.zeros(3, dtype=np.int64)
    for s in range(steps):
        ev = ctx.cascade_step(pops, e, b, dt, 21, s, photon_min_energy=thr)
        r = cas.cascade_step(mid_tables, orc.F64, orc.F64, opops, e, b, dt, 21, s, photon_min_energy=thr)
        assert ev == tuple(r["events"]), (s, ev, r["events"])
        for k in pops:
            assert pops[k].n == opops[k].n, (s, k)
        tot += np.array(ev)
    assert tot[0] > n // 2 and (b0 < 5e-3 or (tot[2] > 20 and tot[1] > 0))
    for k in pops:
        gp, gt = _state(pops[k])
        op, ot = opops[k].p, opops[k].tau
        norm = np.sqrt(sum(a * a for a in op))
        for c in range(3):
            assert np.all(np.abs(gp[c] - op[c]) <= 1e-9 * norm), (k, c)
        dead = norm == 0
        assert np.array_equal(np.isinf(gt), np.isinf(ot)) and np.array_equal(dead, np.sqrt(sum(a * a for a in gp)) == 0)
        live = ~np.isinf(ot)
        assert np.all(np.abs(gt[live] - ot[live]) <= 1e-9 * (np.abs(ot[live]) + 1e-3))
    # spectra of the final state (Fig.6): the GPU histogram of the GPU state equals the oracle histogram of it
    import torch
    for k, species in (("electrons", LEPTON), ("positrons", LEPTON), ("photons", PHOTON)):
        pop = pops[k]
        hist = torch.zeros(60, dtype=torch.int64, device="cuda")
        ctx.energy_spectrum(species, [t[:pop.n] for t in pop.p], 1e-3, 1e3, hist)
        ref, x = cas.energy_spectrum(species, _state(pop)[0], 1e-3, 1e3, 60)
        xs = x[~np.isnan(x)]
        assert np.abs(hist.cpu().numpy() - ref).sum() <= 2 * (np.abs(xs - np.round(xs)) < 1e-9).sum()


@pytest.mark.parametrize("dtype,tdtype", [(np.float32, np.float32), (np.float32, np.float64)])
def test_cascade_fp32_invariants(orc, qed, ctx, cas, dtype, tdtype):
    """single precision (the paper's Fig.6 runs): the loop's bookkeeping and energy conservation; element-wise parity
    of the fp32 QED step itself is test_gpu_parity.py::test_fused_step"""
    n, g0, steps = 4000, 1000.0, 40
    pops, _ = _start(qed, ctx, orc, cas, n, g0, 22, dtype, tdtype, 40 * n)
    e, b = (0.0, 0.0, 0.0), (0.0, 0.0, 9e-3)
    tot = np.zeros(3, dtype=np.int64)
    for s in range(steps):
        before = {k: v.n for k, v in pops.items()}
        ev = ctx.cascade_step(pops, e, b, 1e-16 / steps, 22, s)
        assert pops["photons"].n == before["photons"] + ev[0] + ev[1]
        assert pops["electrons"].n == before["electrons"] + ev[2] and pops["positrons"].n == before["positrons"] + ev[2]
        tot += np.array(ev)
    assert tot[0] > n // 2 and tot[2] > 20
    (ep, _), (pp, _), (gp, gt) = [_state(pops[k]) for k in ("electrons", "positrons", "photons")]
    dead = np.sqrt(sum(a * a for a in gp)) == 0
    assert dead.sum() == tot[2] and np.all(np.isinf(gt[dead])) and np.all(np.isfinite(gt[~dead]))
    total = (np.sqrt(1 + sum(a * a for a in ep)).sum() + np.sqrt(1 + sum(a * a for a in pp)).sum()
             + np.sqrt(sum(a * a for a in gp)).sum())
    assert abs(total / (n * g0) - 1) < 2e-5


def test_cascade_capacity_overflow_is_reported(orc, qed, ctx, cas):
    n = 2000
    pops, _ = _start(qed, ctx, orc, cas, n, 1000.0, 23, np.float64, np.float64, n + 50)
    with pytest.raises(qed.PicsarQedError):
        for s in range(40):
            ctx.cascade_step(pops, (0, 0, 0), (0, 0, 9e-3), 1e-17, 23, s)
    assert pops["photons"].n == pops["photons"].capacity


# ----------------------------------------------------------------------------- chi threshold + classical model
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("n", [70001, 3])
def test_classical_loss_and_threshold(orc, qed, ctx, mid_tables, dtype, n):
    """picsarqed_set_chi_threshold / picsarqed_classical_loss against the oracle: below the threshold the optical depth
    does not move and the momentum shrinks by the classical power; at or above it nothing changes"""
    import torch
    species = LEPTON
    p, e, b = qed.workloads.config1(seed=61, n=n, species=species, dtype=dtype)
    thr, dt = 0.05, 4e-16
    tabs = mid_tables.with_fp32_reads(np.dtype(dtype) == np.float32).with_chi_event_min(thr)
    chi = orc.chi(species, p, e, b)
    near = np.abs(chi - thr) <= 1e-6 * thr                      # (fp32: which side of the threshold is a rounding matter)
    low = (chi < thr) & ~near
    dp, de, db = to_dev(p), to_dev(e), to_dev(b)
    ctx.set_chi_threshold(thr)
    try:
        ctx.classical_loss(dp, de, db, dt)
        got = to_host(dp)
        ref = orc.classical_loss(code(dtype), p, e, b, dt, thr)
        tol = 1e-9 if dtype == np.float64 else 1e-5
        norm = np.sqrt(sum(np.asarray(a, np.float64) ** 2 for a in p))
        for g_, r_, p_ in zip(got, ref, p):
            ok = ~near
            assert np.all(np.abs(g_[ok].astype(np.float64) - r_[ok]) <= tol * norm[ok])
            assert np.array_equal(g_[~low & ~near], p_[~low & ~near])                 # untouched, bit for bit
        if n > 10:
            assert 0.1 * n < low.sum() < 0.9 * n
        # the evolve pass with the threshold: tau of the particles below it does not move
        for sp in (LEPTON, PHOTON):
            p2, e2, b2 = qed.workloads.config1(seed=62, n=n, species=sp, dtype=dtype)
            chi2 = orc.chi(sp, p2, e2, b2)
            tau0 = orc.init_optical_depth(sp, code(dtype), n, 4).astype(dtype)
            dtau = torch.from_numpy(tau0.copy()).cuda()
            ctx.evolve_optical_depth(sp, to_dev(p2), to_dev(e2), to_dev(b2), 1e-15, dtau)
            o = orc.evolve_optical_depth(tabs, sp, code(dtype), p2, e2, b2, 1e-15, tau0)
            g_tau = dtau.cpu().numpy()
            clear = np.abs(chi2 - thr) > 1e-6 * thr
            assert np.array_equal(g_tau[(chi2 < thr) & clear], tau0[(chi2 < thr) & clear])
            fin = clear & np.isfinite(o["tau_exact"])
            assert np.all(np.abs(g_tau[fin].astype(np.float64) - o["tau_exact"][fin]) <= tol * (np.abs(tau0[fin]) + o["decr"][fin]))
    finally:
        ctx.set_chi_threshold(0.0)


def test_cascade_with_chi_threshold_fp64(orc, qed, ctx, cas, mid_tables):
    """the closed loop with the WarpX-side chi threshold: Ridgers case (i) with a threshold above the
    electrons' chi = 1 would switch everything off, so the threshold sits inside the population a cascade produces"""
    n, g0, b0, steps = 3000, 1000.0, 9e-3, 30
    thr = 2.0                                                   # chi_0 = 9: primaries above, most secondaries below
    pops, opops = _start(qed, ctx, orc, cas, n, g0, 23, np.float64, np.float64, 40 * n)
    tabs = mid_tables.with_chi_event_min(thr)
    e, b = (0.0, 0.0, 0.0), (0.0, 0.0, b0)
    dt = 1e-16 / steps
    ctx.set_chi_threshold(thr)
    try:
        for s in range(steps):
            ev = ctx.cascade_step(pops, e, b, dt, 23, s, photon_min_energy=2.0)
            r = cas.cascade_step(tabs, orc.F64, orc.F64, opops, e, b, dt, 23, s, photon_min_energy=2.0)
            assert ev == tuple(r["events"]), (s, ev, r["events"])
    finally:
        ctx.set_chi_threshold(0.0)
    for k in pops:
        assert pops[k].n == opops[k].n
        gp, gt = _state(pops[k])
        op = opops[k].p
        norm = np.sqrt(sum(a * a for a in op))
        for c in range(3):
            assert np.all(np.abs(gp[c] - op[c]) <= 1e-9 * norm), (k, c)
    # the classical model acted: some electrons sit below the threshold and lost energy without emitting
    el_p, _ = _state(pops["electrons"])
    g = np.sqrt(1 + sum(a * a for a in el_p))
    assert (g * b0 < thr).any()


def test_cascade_rejects_overlapping_lepton_id_ranges(qed, ctx):
    """electrons and positrons share the lepton Philox stream: equal id ranges would give pair partners the same draws"""
    import torch
    pops = {k: qed.Species(1024, torch.float64, torch.float64, 0 if k != "photons" else 1 << 41)
            for k in ("electrons", "positrons", "photons")}
    pops["electrons"].n = 8
    with pytest.raises(qed.PicsarQedError):
        ctx.cascade_step(pops, (0.0, 0.0, 0.0), (0.0, 0.0, 1e-3), 1e-17, 1, 0)
