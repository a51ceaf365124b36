"""GPU parity: the CUDA library (through its C ABI) against the CPU oracle, element by element,
on the same seeded inputs and the same table bytes."""
import numpy as np
import pytest

from parity_common import (EPS, F32, F64, LEPTON, PHOTON, TOL_TAU, assert_chi_close, check_evolve, code, to_dev,
                           to_host)

pytestmark = pytest.mark.gpu

DTYPES = [(np.float64, np.float64), (np.float32, np.float32), (np.float32, np.float64)]
IDS = ["f64", "f32", "f32_tau64"]


@pytest.fixture(scope="module")
def qed():
    import paper_2110_00256_b200 as q
    return q


@pytest.fixture(scope="module")
def mid_tables(orc):
    """oracle-built tables, several brackets per decade, built in seconds; C1 ranges"""
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


def _tables_for(mid_tables, dtype):
    return mid_tables.with_fp32_reads(np.dtype(dtype) == np.float32)


def _dt_for(orc, qed, tables, species, p, e, b):
    return qed.workloads.choose_dt(orc.rate(tables, species, p, e, b)[:65536], 0.05)


# ----------------------------------------------------------------------------- chi
@pytest.mark.parametrize("species", [LEPTON, PHOTON])
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("n", [100003, 1, 5])
def test_chi(orc, qed, ctx, species, dtype, n):
    p, e, b = qed.workloads.config1(seed=1, n=n, species=species, dtype=dtype)
    chi_gpu = to_host([ctx.chi(species, to_dev(p), to_dev(e), to_dev(b))])[0]
    chi_orc = orc.chi(species, p, e, b)
    n_cond = assert_chi_close(chi_gpu, chi_orc, species, p, e, b)
    assert n_cond <= max(1, n // 10000)


def test_chi_paper_cases_and_corners(orc, qed, ctx):
    """the paper's worked cases and the cancellation corner e || p"""
    import math
    rows = []
    for g0, bz in ((1000.0, 1e-3), (1000.0, 9e-3)):
        rows.append(((math.sqrt(g0 * g0 - 1), 0, 0), (0, 0, 0), (0, 0, bz)))
    rows.append(((math.sqrt(4120.0 ** 2 - 1), 0, 0), (0, 1.22e-4, 0), (0, 0, -1.22e-4)))
    rows.append(((300.0, 0, 0), (2e-3, 0, 0), (0, 0, 0)))      # e || p: lepton chi = |e|, photon 0
    rows.append(((0.0, 0, 0), (1e-3, 2e-3, 0), (0, 3e-3, 0)))  # p = 0: lepton chi = |e|
    rows += [rows[0]] * 3                                      # pad to a multiple of the vector width
    a = np.array(rows, dtype=np.float64)
    p, e, b = [[np.ascontiguousarray(a[:, k, j]) for j in range(3)] for k in range(3)]
    for sp in (LEPTON, PHOTON):
        got = to_host([ctx.chi(sp, to_dev(p), to_dev(e), to_dev(b))])[0]
        assert_chi_close(got, orc.chi(sp, p, e, b), sp, p, e, b)
    got = to_host([ctx.chi(LEPTON, to_dev(p), to_dev(e), to_dev(b))])[0]
    assert got[0] == pytest.approx(1.0, rel=2e-3) and got[1] == pytest.approx(9.0, rel=2e-3)
    assert got[2] == pytest.approx(1.0, rel=1e-2) and got[3] == pytest.approx(2e-3, rel=1e-14)


# ----------------------------------------------------------------------------- tau = -ln U
@pytest.mark.parametrize("species", [LEPTON, PHOTON])
@pytest.mark.parametrize("tdtype", [np.float64, np.float32])
def test_init_optical_depth(orc, qed, ctx, species, tdtype):
    import torch
    n, seed, id_base = 70001, 11, 5_000_000_000
    tau = torch.empty(n, dtype=torch.float64 if tdtype == np.float64 else torch.float32, device="cuda")
    ctx.init_optical_depth(species, tau, seed, id_base)
    ref = orc.init_optical_depth(species, code(tdtype), n, seed, ids=id_base + np.arange(n, dtype=np.uint64))
    got = tau.cpu().numpy().astype(np.float64)
    assert np.all(np.abs(got - ref) <= 4 * EPS[np.dtype(tdtype)] * np.abs(ref))
    assert np.all(got > 0) and np.all(np.isfinite(got))


# ----------------------------------------------------------------------------- evolve
@pytest.mark.parametrize("species", [LEPTON, PHOTON])
@pytest.mark.parametrize("dtype,tdtype", DTYPES, ids=IDS)
@pytest.mark.parametrize("n", [65536 + 37, 3])
def test_evolve(orc, qed, ctx, mid_tables, species, dtype, tdtype, n):
    import torch
    p, e, b = qed.workloads.config1(seed=1, n=n, species=species, dtype=dtype)
    tables = _tables_for(mid_tables, dtype)
    dt = _dt_for(orc, qed, tables, species, p, e, b)
    tau0 = orc.init_optical_depth(species, code(tdtype), n, 1).astype(tdtype)
    if species == PHOTON and n > 100:
        tau0[17] = np.inf  # a dead photon stays dead
    tau = torch.from_numpy(tau0.copy()).cuda()
    count = torch.zeros(1, dtype=torch.int64, device="cuda")
    ctx.evolve_optical_depth(species, to_dev(p), to_dev(e), to_dev(b), dt, tau, count)
    o = orc.evolve_optical_depth(tables, species, code(tdtype), p, e, b, dt, tau0)
    ln_chi = np.log(np.maximum(orc.chi(species, p, e, b), 1e-300))
    n_amb, flags = check_evolve(tau.cpu().numpy(), tau0.astype(np.float64), o, dtype, ln_chi)
    assert ctx.read_count(count) == int(flags.sum())
    assert n_amb <= (0 if dtype == np.float64 else 3)
    if n > 100:
        assert 0.02 < flags.mean() < 0.1  # the 5 % rule


def test_evolve_erber_branches_and_table_edges(orc, qed, ctx, mid_tables):
    """photons below / above the T table use eq.10; leptons clamp"""
    import torch
    chi_t = np.array([1e-5, 1e-3, 5e-3, 0.019, 0.021, 1.0, 999.0, 1001.0, 5e3, 1e5, 0.2, 30.0])
    n = chi_t.size
    g = 2000.0
    for sp in (LEPTON, PHOTON):
        pm = np.sqrt(g * g - 1) if sp == LEPTON else g
        p = [np.full(n, pm), np.zeros(n), np.zeros(n)]
        e = [np.zeros(n)] * 3
        b = [np.zeros(n), np.zeros(n), chi_t / pm]
        tau0 = np.full(n, 0.3)
        dt = 0.05 / orc.rate(mid_tables, sp, p, e, b)[5]
        tau = torch.from_numpy(tau0.copy()).cuda()
        ctx.evolve_optical_depth(sp, to_dev(p), to_dev(e), to_dev(b), dt, tau)
        o = orc.evolve_optical_depth(mid_tables, sp, F64, p, e, b, dt, tau0)
        got = tau.cpu().numpy()
        assert np.all(np.abs(got - o["tau_exact"]) <= 1e-9 * (0.3 + o["decr"])), (sp, got - o["tau_exact"])
        # the decrement itself, where it is not negligible
        big = o["decr"] > 1e-6
        assert np.allclose((0.3 - got)[big], o["decr"][big], rtol=1e-8)


def test_evolve_low_energy_photons_never_decay(orc, qed, ctx):
    import torch
    n = 8
    p = [np.array([0.0, 1.0, 1.9, 2.0, 2.0000001, 3.0, 10.0, 100.0]), np.zeros(n), np.zeros(n)]
    e = [np.zeros(n)] * 3
    b = [np.zeros(n), np.zeros(n), np.full(n, 0.5)]
    tau = torch.full((n,), 0.25, dtype=torch.float64, device="cuda")
    ctx.evolve_optical_depth(PHOTON, to_dev(p), to_dev(e), to_dev(b), 1e-15, tau)
    got = tau.cpu().numpy()
    assert np.all(got[:4] == 0.25) and np.all(got[4:] < 0.25)  # gamma_gamma <= 2 cannot decay (R12)


# ----------------------------------------------------------------------------- events
def _vec_close(got, ref, tol):
    """per-component error relative to the vector norm"""
    got = [np.asarray(a, np.float64) for a in got]
    ref = [np.asarray(a, np.float64) for a in ref]
    norm = np.sqrt(sum(a * a for a in ref))
    for g_, r_ in zip(got, ref):
        bad = np.nonzero(~(np.abs(g_ - r_) <= tol * norm))[0]
        assert bad.size == 0, "vector mismatch at %s: %s vs %s (|v| %s)" % (bad[:5], g_[bad[:5]], r_[bad[:5]], norm[bad[:5]])


def _run_events(orc, qed, ctx, tables, species, dtype, tdtype, p, e, b, tau_host, seed, step, id_base, capacity):
    """GPU and oracle event generation on identical inputs; returns (gpu dict, oracle dict)"""
    import torch
    n = tau_host.size
    tdt = torch.float64 if tdtype == np.float64 else torch.float32
    pdt = torch.float64 if dtype == np.float64 else torch.float32
    dp, de, db = to_dev(p), to_dev(e), to_dev(b)
    dtau = torch.from_numpy(tau_host.copy()).cuda()
    nsec = 1 if species == LEPTON else 2
    sec_p = [[torch.full((max(capacity, 1),), -7.0, dtype=pdt, device="cuda") for _ in range(3)] for _ in range(nsec)]
    sec_tau = [torch.full((max(capacity, 1),), -7.0, dtype=tdt, device="cuda") for _ in range(nsec)]
    parent = torch.full((max(capacity, 1),), -1, dtype=torch.int64, device="cuda")
    n_out = torch.zeros(1, dtype=torch.int64, device="cuda")
    ids = id_base + np.arange(n, dtype=np.uint64)
    if species == LEPTON:
        ctx.generate_photons(dp, de, db, dtau, seed, step, id_base, capacity, sec_p[0], sec_tau[0], parent, n_out)
        o = orc.generate_photons(tables, code(dtype), code(tdtype), p, e, b, tau_host, seed, step, ids, capacity)
        o_sec_p, o_sec_tau = [o["ph_p"]], [o["ph_tau"]]
    else:
        ctx.generate_pairs(dp, de, db, dtau, seed, step, id_base, capacity, sec_p[0], sec_tau[0], sec_p[1],
                           sec_tau[1], parent, n_out)
        o = orc.generate_pairs(tables, code(dtype), code(tdtype), p, e, b, tau_host, seed, step, ids, capacity)
        o_sec_p, o_sec_tau = [o["el_p"], o["po_p"]], [o["el_tau"], o["po_tau"]]
    g = dict(n_fired=ctx.read_count(n_out), p=to_host(dp), tau=dtau.cpu().numpy(), parent=parent.cpu().numpy(),
             sec_p=[to_host(s) for s in sec_p], sec_tau=to_host(sec_tau))
    o["sec_p"], o["sec_tau"] = o_sec_p, o_sec_tau
    return g, o


def _compare_events(g, o, species, dtype, tdtype, capacity, p_before):
    tol = TOL_TAU[np.dtype(dtype)]
    ttol = TOL_TAU[np.dtype(tdtype)]
    k = min(o["n_fired"], capacity)
    assert g["n_fired"] == o["n_fired"]                       # bit-exact count
    assert np.array_equal(g["parent"][:k], o["parent"])       # bit-exact compaction order
    assert np.all(np.diff(g["parent"][:k]) > 0)
    for s in range(len(o["sec_p"])):
        _vec_close([a[:k] for a in g["sec_p"][s]], o["sec_p"][s], tol)
        assert np.all(np.abs(g["sec_tau"][s][:k].astype(np.float64) - o["sec_tau"][s]) <= ttol * o["sec_tau"][s])
        for a in g["sec_p"][s]:                               # nothing written past the count
            assert np.all(a[k:] == -7.0)
    # parents: momenta and optical depth rewritten; everything else untouched, bit for bit
    if species == LEPTON:
        _vec_close(g["p"], o["p"], tol)
    else:
        for a, r_ in zip(g["p"], o["p"]):
            assert np.array_equal(a.astype(np.float64), r_)
    untouched = np.ones(g["tau"].size, bool)
    untouched[o["parent"]] = False
    for a, r_ in zip(g["p"], p_before):
        assert np.array_equal(a[untouched], r_[untouched])
    fin = np.isfinite(o["tau"])
    assert np.array_equal(np.isfinite(g["tau"]), fin)
    assert np.all(np.abs(g["tau"][fin].astype(np.float64) - o["tau"][fin]) <= ttol * np.abs(o["tau"][fin]))


@pytest.mark.parametrize("species", [LEPTON, PHOTON])
@pytest.mark.parametrize("dtype,tdtype", DTYPES, ids=IDS)
def test_events(orc, qed, ctx, mid_tables, species, dtype, tdtype):
    n = 3 * 4096 + 1234  # several compaction tiles and a ragged tail
    p, e, b = qed.workloads.config1(seed=4, n=n, species=species, dtype=dtype)
    tables = _tables_for(mid_tables, dtype)
    rng = np.random.default_rng(5)
    tau = rng.exponential(size=n).astype(tdtype)
    fired = rng.uniform(size=n) < 0.07
    fired[:40] = True                # a dense run of events
    fired[4096 * 2:4096 * 3] = False  # an empty tile
    fired[-1] = True
    tau[fired] *= -1
    g, o = _run_events(orc, qed, ctx, tables, species, dtype, tdtype, p, e, b, tau, 21, 3, 1 << 33, n)
    assert o["n_fired"] == int(fired.sum())
    _compare_events(g, o, species, dtype, tdtype, n, p)


@pytest.mark.parametrize("species", [LEPTON, PHOTON])
def test_events_with_2d_tables_on_their_own_row_grid(orc, qed, species):
    """picsarqed_table_params.qs_n_chi_2d / bw_n_chi_2d (BASELINE config 4's shape): the 1D lookups use the 1D grid, the
    row interpolation of eq.24/28 the 2D grid; GPU-built tables, their bytes given to the oracle"""
    kw = dict(qs_chi_min=1e-3, qs_chi_max=1e3, qs_n_chi=64, qs_xi_min=1e-12, qs_n_xi=72,
              bw_chi_min=2e-2, bw_chi_max=1e3, bw_n_chi=48, bw_n_xi=56, qs_n_chi_2d=23, bw_n_chi_2d=31)
    c = qed.Context(0)
    c.build_tables(qed.TableParams(**kw))
    tabs = orc.Tables(orc.TableParams(**kw), c.export_tables(qed.TAB_LNG), c.export_tables(qed.TAB_QS_LNP),
                      c.export_tables(qed.TAB_LNT), c.export_tables(qed.TAB_BW_P))
    n = 2 * 4096 + 321
    p, e, b = qed.workloads.config1(seed=14, n=n, species=species, dtype=np.float64)
    dt = _dt_for(orc, qed, tabs, species, p, e, b)
    tau0 = orc.init_optical_depth(species, F64, n, 3)
    import torch
    dtau = torch.from_numpy(tau0.copy()).cuda()
    c.evolve_optical_depth(species, to_dev(p), to_dev(e), to_dev(b), 3 * dt, dtau)
    o = orc.evolve_optical_depth(tabs, species, F64, p, e, b, 3 * dt, tau0)
    ln_chi = np.log(np.maximum(orc.chi(species, p, e, b), 1e-300))
    tau_mid = dtau.cpu().numpy()
    check_evolve(tau_mid, tau0, o, np.float64, ln_chi)
    g, oe = _run_events(orc, qed, c, tabs, species, np.float64, np.float64, p, e, b, tau_mid, 5, 1, 77, n)
    assert oe["n_fired"] > 200
    _compare_events(g, oe, species, np.float64, np.float64, n, p)
    c.close()


@pytest.mark.parametrize("species", [LEPTON, PHOTON])
@pytest.mark.parametrize("dtype,tdtype", DTYPES, ids=IDS)
def test_views_offset_by_16_bytes(orc, qed, ctx, mid_tables, species, dtype, tdtype):
    """the ABI asks for 16-byte alignment only: every array is a view that starts 16 bytes into its allocation
    (fp32 particles with an fp64 optical depth used to store tau with one 256-bit instruction)"""
    import torch
    n = 3 * 4096 + 50
    off_p = 16 // np.dtype(dtype).itemsize
    off_t = 16 // np.dtype(tdtype).itemsize
    p, e, b = qed.workloads.config1(seed=15, n=n, species=species, dtype=dtype)
    tables = _tables_for(mid_tables, dtype)
    dt = 2 * _dt_for(orc, qed, tables, species, p, e, b)

    def view(a, off):
        buf = torch.zeros(a.size + off + 8, dtype=torch.from_numpy(a[:1]).dtype, device="cuda")
        v = buf[off:off + a.size]
        v.copy_(torch.from_numpy(np.ascontiguousarray(a)))
        assert v.data_ptr() % 32 == 16
        return v

    tau0 = orc.init_optical_depth(species, code(tdtype), n, 9).astype(tdtype)
    for fused in (False, True):
        dp, de, db = [view(a, off_p) for a in p], [view(a, off_p) for a in e], [view(a, off_p) for a in b]
        dtau = view(tau0, off_t)
        nsec = 1 if species == LEPTON else 2
        sec_p = [[view(np.zeros(n, dtype), off_p) for _ in range(3)] for _ in range(nsec)]
        sec_t = [view(np.zeros(n, tdtype), off_t) for _ in range(nsec)]
        n_out = torch.zeros(1, dtype=torch.int64, device="cuda")
        if fused:
            ctx.qed_step(species, dp, de, db, dtau, dt, 1, 0, 0, n, sec_p[0], sec_t[0], sec_p[1] if nsec == 2 else None,
                         sec_t[1] if nsec == 2 else None, None, n_out)
            k = ctx.read_count(n_out)
            assert k == int((tau_mid < 0).sum())
        else:
            ctx.evolve_optical_depth(species, dp, de, db, dt, dtau)
            tau_mid = dtau.cpu().numpy()
            o = orc.evolve_optical_depth(tables, species, code(tdtype), p, e, b, dt, tau0)
            check_evolve(tau_mid, tau0.astype(np.float64), o, dtype, np.log(np.maximum(orc.chi(species, p, e, b), 1e-300)))


@pytest.mark.parametrize("species", [LEPTON, PHOTON])
def test_events_capacity_rule(orc, qed, ctx, mid_tables, species):
    """only the first `capacity` fired parents are processed; the rest keep tau < 0"""
    n = 2 * 4096 + 77
    p, e, b = qed.workloads.config1(seed=6, n=n, species=species, dtype=np.float64)
    rng = np.random.default_rng(7)
    tau = np.where(rng.uniform(size=n) < 0.1, -0.5, 0.5)
    total = int((tau < 0).sum())
    for cap in (0, 1, 300, total, total + 5):
        g, o = _run_events(orc, qed, ctx, mid_tables, species, np.float64, np.float64, p, e, b, tau, 1, 0, 0, cap)
        assert g["n_fired"] == total
        _compare_events(g, o, species, np.float64, np.float64, cap, p)
        late = np.nonzero(tau < 0)[0][cap:]
        assert np.all(g["tau"][late] == -0.5)


@pytest.mark.parametrize("species", [LEPTON, PHOTON])
def test_events_degenerate(orc, qed, ctx, mid_tables, species):
    """no events, all events, n = 1"""
    for n, frac in ((5000, 0.0), (4096 + 5, 1.0), (1, 1.0), (1, 0.0)):
        p, e, b = qed.workloads.config1(seed=8, n=n, species=species, dtype=np.float64)
        tau = np.full(n, 0.4) if frac == 0.0 else np.full(n, -0.4)
        g, o = _run_events(orc, qed, ctx, mid_tables, species, np.float64, np.float64, p, e, b, tau, 2, 9, 100, n)
        assert g["n_fired"] == (n if frac else 0)
        _compare_events(g, o, species, np.float64, np.float64, n, p)


def test_empty_inputs(qed, ctx):
    import torch
    z = [torch.empty(0, dtype=torch.float64, device="cuda") for _ in range(3)]
    tau = torch.empty(0, dtype=torch.float64, device="cuda")
    cnt = torch.full((1,), 99, dtype=torch.int64, device="cuda")
    ctx.evolve_optical_depth(LEPTON, z, z, z, 1e-15, tau, cnt)
    assert ctx.read_count(cnt) == 0
    cnt.fill_(99)
    ctx.generate_photons(z, z, z, tau, 1, 0, 0, 0, z, tau, None, cnt)
    assert ctx.read_count(cnt) == 0
    assert ctx.chi(LEPTON, z, z, z).numel() == 0


# ----------------------------------------------------------------------------- multi-step, free running
@pytest.mark.parametrize("species,dtype,tdtype", [(LEPTON, np.float64, np.float64), (PHOTON, np.float32, np.float32),
                                                  (LEPTON, np.float32, np.float64)], ids=["qs_f64", "bw_f32", "qs_mixed"])
def test_free_running_steps(orc, qed, ctx, mid_tables, species, dtype, tdtype):
    """evolve + events for several steps on both sides; the oracle adopts the GPU flag only for
    particles inside the tie margin"""
    import torch
    n, steps, seed = 20000 + 3, 4, 13
    p, e, b = qed.workloads.config1(seed=9, n=n, species=species, dtype=dtype)
    tables = _tables_for(mid_tables, dtype)
    dt = _dt_for(orc, qed, tables, species, p, e, b)
    tau_h = orc.init_optical_depth(species, code(tdtype), n, seed).astype(tdtype)
    dp, de, db = to_dev(p), to_dev(e), to_dev(b)
    dtau = torch.from_numpy(tau_h.copy()).cuda()
    p_h = [a.copy() for a in p]
    total_amb = 0
    for step in range(steps):
        ctx.evolve_optical_depth(species, dp, de, db, dt, dtau)
        o = orc.evolve_optical_depth(tables, species, code(tdtype), p_h, e, b, dt, tau_h)
        ln_chi = np.log(np.maximum(orc.chi(species, p_h, e, b), 1e-300))
        tau_gpu = dtau.cpu().numpy()
        n_amb, flags = check_evolve(tau_gpu, tau_h.astype(np.float64), o, dtype, ln_chi)
        total_amb += n_amb
        # both sides continue from the GPU's tau (differences are within tolerance; flags are the GPU's)
        g, oe = _run_events(orc, qed, ctx, tables, species, dtype, tdtype, p_h, e, b, tau_gpu, seed, step, 0, n)
        _compare_events(g, oe, species, dtype, tdtype, n, p_h)
        p_h, tau_h = g["p"], g["tau"]
        dp, dtau = to_dev(p_h), torch.from_numpy(tau_h.copy()).cuda()
    assert total_amb <= (0 if dtype == np.float64 else 5)


# ----------------------------------------------------------------------------- fused step
def _run_fused(qed, ctx, species, dtype, tdtype, p, e, b, tau_host, dt, seed, step, id_base, capacity):
    import torch
    tdt = torch.float64 if tdtype == np.float64 else torch.float32
    pdt = torch.float64 if dtype == np.float64 else torch.float32
    dp, de, db = to_dev(p), to_dev(e), to_dev(b)
    dtau = torch.from_numpy(tau_host.copy()).cuda()
    nsec = 1 if species == LEPTON else 2
    cap = max(capacity, 1)
    sec_p = [[torch.full((cap,), -7.0, dtype=pdt, device="cuda") for _ in range(3)] for _ in range(nsec)]
    sec_tau = [torch.full((cap,), -7.0, dtype=tdt, device="cuda") for _ in range(nsec)]
    parent = torch.full((cap,), -1, dtype=torch.int64, device="cuda")
    n_out = torch.zeros(1, dtype=torch.int64, device="cuda")
    ctx.qed_step(species, dp, de, db, dtau, dt, seed, step, id_base, capacity, sec_p[0], sec_tau[0],
                 sec_p[1] if nsec == 2 else None, sec_tau[1] if nsec == 2 else None, parent, n_out)
    return dict(n_fired=ctx.read_count(n_out), p=to_host(dp), tau=dtau.cpu().numpy(), parent=parent.cpu().numpy(),
                sec_p=[to_host(s) for s in sec_p], sec_tau=to_host(sec_tau))


def _run_unfused(qed, ctx, species, dtype, tdtype, p, e, b, tau_host, dt, seed, step, id_base, capacity):
    import torch
    tdt = torch.float64 if tdtype == np.float64 else torch.float32
    pdt = torch.float64 if dtype == np.float64 else torch.float32
    dp, de, db = to_dev(p), to_dev(e), to_dev(b)
    dtau = torch.from_numpy(tau_host.copy()).cuda()
    nsec = 1 if species == LEPTON else 2
    cap = max(capacity, 1)
    sec_p = [[torch.full((cap,), -7.0, dtype=pdt, device="cuda") for _ in range(3)] for _ in range(nsec)]
    sec_tau = [torch.full((cap,), -7.0, dtype=tdt, device="cuda") for _ in range(nsec)]
    parent = torch.full((cap,), -1, dtype=torch.int64, device="cuda")
    n_out = torch.zeros(1, dtype=torch.int64, device="cuda")
    ctx.evolve_optical_depth(species, dp, de, db, dt, dtau)
    tau_mid = dtau.cpu().numpy()
    if species == LEPTON:
        ctx.generate_photons(dp, de, db, dtau, seed, step, id_base, capacity, sec_p[0], sec_tau[0], parent, n_out)
    else:
        ctx.generate_pairs(dp, de, db, dtau, seed, step, id_base, capacity, sec_p[0], sec_tau[0], sec_p[1], sec_tau[1],
                           parent, n_out)
    return dict(n_fired=ctx.read_count(n_out), p=to_host(dp), tau=dtau.cpu().numpy(), parent=parent.cpu().numpy(),
                sec_p=[to_host(s) for s in sec_p], sec_tau=to_host(sec_tau)), tau_mid


def _same(a, b):
    return np.array_equal(a, b, equal_nan=True)


@pytest.mark.parametrize("species", [LEPTON, PHOTON])
@pytest.mark.parametrize("dtype,tdtype", DTYPES, ids=IDS)
@pytest.mark.parametrize("n,target", [(5 * 4096 + 1234, 0.05), (4096 + 77, 0.6), (1000, 0.05), (1, 0.9)])
def test_fused_step(orc, qed, ctx, mid_tables, species, dtype, tdtype, n, target):
    """picsarqed_qed_step == evolve followed by generate, bit for bit (same device functions), and both agree with the
    oracle; target 0.6 overflows the shared-memory record buffer (more than a quarter of a tile fires)"""
    p, e, b = qed.workloads.config1(seed=31, n=n, species=species, dtype=dtype)
    tables = _tables_for(mid_tables, dtype)
    dt = qed.workloads.choose_dt(orc.rate(tables, species, p, e, b), target)
    tau0 = orc.init_optical_depth(species, code(tdtype), n, 5).astype(tdtype)
    for cap in (n, max(1, n // 40)):
        f = _run_fused(qed, ctx, species, dtype, tdtype, p, e, b, tau0, dt, 77, 2, 123456789, cap)
        u, tau_mid = _run_unfused(qed, ctx, species, dtype, tdtype, p, e, b, tau0, dt, 77, 2, 123456789, cap)
        # the two calls again with "stage_records": evolve_optical_depth stages what generate_* then takes
        ctx.set_option("stage_records", 1)
        try:
            u2, tau_mid2 = _run_unfused(qed, ctx, species, dtype, tdtype, p, e, b, tau0, dt, 77, 2, 123456789, cap)
        finally:
            ctx.set_option("stage_records", 0)
        assert _same(tau_mid, tau_mid2)
        for other in (u, u2):
            assert f["n_fired"] == other["n_fired"] and _same(f["parent"], other["parent"])
            assert _same(f["tau"], other["tau"]) and all(_same(x, y) for x, y in zip(f["p"], other["p"]))
            for s in range(len(f["sec_p"])):
                assert all(_same(x, y) for x, y in zip(f["sec_p"][s], other["sec_p"][s]))
                assert _same(f["sec_tau"][s], other["sec_tau"][s])
        # and against the oracle: evolve with the tie protocol, events on the GPU's evolved tau
        o = orc.evolve_optical_depth(tables, species, code(tdtype), p, e, b, dt, tau0)
        ln_chi = np.log(np.maximum(orc.chi(species, p, e, b), 1e-300))
        check_evolve(tau_mid, tau0.astype(np.float64), o, dtype, ln_chi)
        ids = 123456789 + np.arange(n, dtype=np.uint64)
        if species == LEPTON:
            oe = orc.generate_photons(tables, code(dtype), code(tdtype), p, e, b, tau_mid, 77, 2, ids, cap)
            oe["sec_p"], oe["sec_tau"] = [oe["ph_p"]], [oe["ph_tau"]]
        else:
            oe = orc.generate_pairs(tables, code(dtype), code(tdtype), p, e, b, tau_mid, 77, 2, ids, cap)
            oe["sec_p"], oe["sec_tau"] = [oe["el_p"], oe["po_p"]], [oe["el_tau"], oe["po_tau"]]
        _compare_events(f, oe, species, dtype, tdtype, cap, p)
        if n > 4096:
            assert f["n_fired"] > 0.5 * target * n


@pytest.mark.parametrize("species", [LEPTON, PHOTON])
@pytest.mark.parametrize("dtype,tdtype", DTYPES, ids=IDS)
@pytest.mark.parametrize("config", [0, 1])
def test_fused_kernel_matches_the_two_kernel_step(orc, qed, ctx, mid_tables, species, dtype, tdtype, config):
    """option "fused_step" (step.cuh: TMA-staged streaming warps + event warps, parents rewritten while their sectors are in
    L2): bit for bit what the default evolve pass + event pass give -- all tiles, a ragged end, chunks with more than 24
    events, a capacity below the number of events (the undo path of the placement), both register configurations"""
    for n, target in ((9 * 2048 + 777, 0.06), (2 * 2048 + 5, 0.5), (300, 0.06)):
        p, e, b = qed.workloads.config1(seed=51, n=n, species=species, dtype=dtype)
        tables = _tables_for(mid_tables, dtype)
        dt = qed.workloads.choose_dt(orc.rate(tables, species, p, e, b), target)
        tau0 = orc.init_optical_depth(species, code(tdtype), n, 7).astype(tdtype)
        for cap in (n, max(1, n // 50)):
            ref = _run_fused(qed, ctx, species, dtype, tdtype, p, e, b, tau0, dt, 5, 3, 1 << 35, cap)
            ctx.set_option("fused_step", 1)
            ctx.set_option("step_config", config)
            try:
                got = _run_fused(qed, ctx, species, dtype, tdtype, p, e, b, tau0, dt, 5, 3, 1 << 35, cap)
            finally:
                ctx.set_option("fused_step", 0)
                ctx.set_option("step_config", 0)
            assert got["n_fired"] == ref["n_fired"] and _same(got["parent"], ref["parent"])
            assert _same(got["tau"], ref["tau"]) and all(_same(x, y) for x, y in zip(got["p"], ref["p"]))
            for s_ in range(len(ref["sec_p"])):
                assert all(_same(x, y) for x, y in zip(got["sec_p"][s_], ref["sec_p"][s_]))
                assert _same(got["sec_tau"][s_], ref["sec_tau"][s_])
            if n > 2048:
                assert ref["n_fired"] > 0.5 * target * n


@pytest.mark.parametrize("dtype,tdtype", DTYPES, ids=IDS)
def test_optical_depth_redrawn_by_either_pass(orc, qed, ctx, mid_tables, dtype, tdtype):
    """option "evolve_redraw": whether the evolve pass (one Philox pass per chunk, the new value leaves with the pass's vector store)
    or the event pass (a fourth scattered store) re-draws the optical depth of the leptons that emit, every output is the same bit
    for bit -- all tiles, a ragged end, chunks with more than 24 events (which the event pass re-scans: their parents are re-drawn
    there), and a capacity below the number of events: the parents beyond it keep their evolved, negative optical depth"""
    for n, target in ((9 * 2048 + 777, 0.06), (2 * 2048 + 5, 0.5), (300, 0.06)):
        p, e, b = qed.workloads.config1(seed=61, n=n, species=LEPTON, dtype=dtype)
        tables = _tables_for(mid_tables, dtype)
        dt = qed.workloads.choose_dt(orc.rate(tables, LEPTON, p, e, b), target)
        tau0 = orc.init_optical_depth(LEPTON, code(tdtype), n, 9).astype(tdtype)
        for cap in (n, max(1, n // 50)):
            runs = []
            for mode in (0, 1, 2):
                ctx.set_option("evolve_redraw", mode)
                try:
                    runs.append(_run_fused(qed, ctx, LEPTON, dtype, tdtype, p, e, b, tau0, dt, 5, 3, 1 << 35, cap))
                finally:
                    ctx.set_option("evolve_redraw", 2)
            ref = runs[0]
            for got in runs[1:]:
                assert got["n_fired"] == ref["n_fired"] and _same(got["parent"], ref["parent"])
                assert _same(got["tau"], ref["tau"]) and all(_same(x, y) for x, y in zip(got["p"], ref["p"]))
                assert all(_same(x, y) for x, y in zip(got["sec_p"][0], ref["sec_p"][0]))
                assert _same(got["sec_tau"][0], ref["sec_tau"][0])
            if cap < ref["n_fired"]:
                assert int((ref["tau"] < 0).sum()) == ref["n_fired"] - cap     # the parents beyond the capacity wait, untouched


def test_staged_records_are_dropped_when_not_consumed(orc, qed, ctx, mid_tables):
    """"stage_records": records staged by an evolve call that no generate call consumes (another evolve, another array,
    another size in between) must not leak into the next event pass"""
    import torch
    n = 2 * 4096 + 300
    p, e, b = qed.workloads.config1(seed=41, n=n, species=LEPTON, dtype=np.float64)
    dt = 3 * qed.workloads.choose_dt(orc.rate(mid_tables, LEPTON, p, e, b), 0.05)
    tau0 = orc.init_optical_depth(LEPTON, F64, n, 6)
    ref, _ = _run_unfused(qed, ctx, LEPTON, np.float64, np.float64, p, e, b, tau0, dt, 3, 1, 0, n)
    ctx.set_option("stage_records", 1)
    try:
        dp, de, db = to_dev(p), to_dev(e), to_dev(b)
        other = torch.from_numpy(tau0.copy()).cuda()
        ctx.evolve_optical_depth(LEPTON, dp, de, db, 5 * dt, other)                 # staged, never consumed
        ctx.evolve_optical_depth(LEPTON, [t[:4096] for t in dp], [t[:4096] for t in de], [t[:4096] for t in db], dt,
                                 torch.from_numpy(tau0[:4096].copy()).cuda())        # another size
        got, _ = _run_unfused(qed, ctx, LEPTON, np.float64, np.float64, p, e, b, tau0, dt, 3, 1, 0, n)
        # a generate call on an array that was NOT the last one evolved re-scans tau
        dtau = torch.from_numpy(tau0.copy()).cuda()
        ctx.evolve_optical_depth(LEPTON, dp, de, db, dt, dtau)
        ctx.evolve_optical_depth(LEPTON, dp, de, db, 5 * dt, other)
        sec_p = [torch.zeros(n, dtype=torch.float64, device="cuda") for _ in range(3)]
        sec_t = torch.zeros(n, dtype=torch.float64, device="cuda")
        parent = torch.full((n,), -1, dtype=torch.int64, device="cuda")
        n_out = torch.zeros(1, dtype=torch.int64, device="cuda")
        ctx.generate_photons(dp, de, db, dtau, 3, 1, 0, n, sec_p, sec_t, parent, n_out)
        k = ctx.read_count(n_out)
    finally:
        ctx.set_option("stage_records", 0)
    assert got["n_fired"] == ref["n_fired"] and _same(got["parent"], ref["parent"]) and _same(got["tau"], ref["tau"])
    assert k == ref["n_fired"] and _same(parent.cpu().numpy(), ref["parent"]) and _same(dtau.cpu().numpy(), ref["tau"])


def test_fused_step_repeated_launches(qed, ctx):
    """many launches back to back on one context: the ticket counter and the epoch-stamped status words carry over"""
    import torch
    n = 3 * 4096 + 5
    p, e, b = qed.workloads.config1(seed=32, n=n, species=LEPTON, dtype=np.float64)
    dp, de, db = to_dev(p), to_dev(e), to_dev(b)
    tau = torch.full((n,), 0.01, dtype=torch.float64, device="cuda")
    sec_p = [torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3)]
    sec_tau = torch.empty(n, dtype=torch.float64, device="cuda")
    n_out = torch.zeros(1, dtype=torch.int64, device="cuda")
    counts = []
    for step in range(40):
        sec_tau.fill_(-7.0)
        ctx.qed_step(LEPTON, dp, de, db, tau, 3e-18, 1, step, 0, n, sec_p, sec_tau, None, None, None, n_out)
        k = ctx.read_count(n_out)
        counts.append(k)
        assert k == int((sec_tau != -7.0).sum().item()) and bool((sec_tau[:k] > 0).all())  # dense, nothing past the count
        assert bool((tau >= 0).all())                                                      # every fired parent was re-drawn
    assert sum(counts) > 0


@pytest.mark.parametrize("species", [LEPTON, PHOTON])
@pytest.mark.parametrize("dtype,tdtype", [(np.float64, np.float64), (np.float32, np.float32), (np.float32, np.float64)])
def test_step_host_pipeline(orc, qed, ctx, mid_tables, species, dtype, tdtype):
    """picsarqed_step_host (host buffers, slabs pipelined over three streams and chained through device counters)
    == one picsarqed_qed_step over the whole array, bit for bit: momenta, optical depths, secondaries, their
    order, global parent indices, the count and the capacity rule across slab borders.  qed_step itself is held
    to the oracle on these inputs by test_fused_step."""
    import torch
    pdt = torch.float64 if dtype == np.float64 else torch.float32
    tdt = torch.float64 if tdtype == np.float64 else torch.float32
    nsec = 1 if species == LEPTON else 2
    try:
        for n in (3 * 4096 + 77, 8192, 300):
            p, e, b = qed.workloads.config1(seed=33, n=n, species=species, dtype=dtype)
            tables = _tables_for(mid_tables, dtype)
            dt = qed.workloads.choose_dt(orc.rate(tables, species, p, e, b), 0.2)
            tau0 = orc.init_optical_depth(species, code(tdtype), n, 6).astype(tdtype)
            for cap in (n, max(1, n // 40)):
                f = _run_fused(qed, ctx, species, dtype, tdtype, p, e, b, tau0, dt, 78, 3, 987654321, cap)
                m = min(f["n_fired"], cap)
                assert f["n_fired"] > cap or cap == n
                for slabs in (0, 1, 3, 7):
                    ctx.set_option("host_slabs", slabs)
                    hp = [torch.from_numpy(np.ascontiguousarray(x)).pin_memory() for x in p]
                    he = [torch.from_numpy(np.ascontiguousarray(x)).pin_memory() for x in e]
                    hb = [torch.from_numpy(np.ascontiguousarray(x)).pin_memory() for x in b]
                    htau = torch.from_numpy(tau0.copy()).pin_memory()
                    sec = [torch.full((cap,), -7.0, dtype=tdt if k % 4 == 3 else pdt).pin_memory() for k in range(4 * nsec)]
                    parent = torch.full((cap,), -1, dtype=torch.int64).pin_memory()
                    fired = ctx.step_host(species, hp, he, hb, htau, dt, 78, 3, 987654321, cap, sec, parent)
                    assert fired == f["n_fired"], (n, cap, slabs)
                    assert _same(htau.numpy(), f["tau"]) and all(_same(x.numpy(), y) for x, y in zip(hp, f["p"]))
                    assert _same(parent.numpy()[:m], f["parent"][:m]) and bool((parent[m:] == -1).all())
                    for s_ in range(nsec):
                        for k in range(3):
                            assert _same(sec[4 * s_ + k].numpy()[:m], f["sec_p"][s_][k][:m])
                        assert _same(sec[4 * s_ + 3].numpy()[:m], f["sec_tau"][s_][:m])
                        assert bool((sec[4 * s_ + 3][m:] == -7.0).all())
    finally:
        ctx.set_option("host_slabs", 0)


@pytest.mark.parametrize("species", [LEPTON, PHOTON])
def test_evolve_decrement_accuracy_fp64(orc, qed, ctx, mid_tables, species):
    """the decrement itself (tau_old = 0), far tighter than the 1e-9 of the north star: the kernel uses its own lean
    log/exp/rcp/rsqrt, whose errors must stay at the few-ulp level; the bound is the conditioning of the lookup"""
    import torch
    n = 50000
    p, e, b = qed.workloads.config1(seed=41, n=n, species=species)
    dt = 1e-17
    tau = torch.zeros(n, dtype=torch.float64, device="cuda")
    ctx.evolve_optical_depth(species, to_dev(p), to_dev(e), to_dev(b), dt, tau)
    o = orc.evolve_optical_depth(mid_tables, species, F64, p, e, b, dt, np.zeros(n))
    d_gpu, d_orc = -tau.cpu().numpy(), o["decr"]
    ln_chi = np.log(np.maximum(orc.chi(species, p, e, b), 1e-300))
    ok = d_orc > 1e-80   # below: photons far under the T table, where the kernel returns exactly 0 (K^2 < e^-200)
    rel = np.abs(d_gpu[ok] - d_orc[ok]) / d_orc[ok]
    from parity_common import uncancelled_scale
    chi_cond = uncancelled_scale(species, p, e, b)[ok] / np.exp(ln_chi[ok])       # conditioning of eq.2 itself
    bound = 2.2e-16 * (32 + np.abs(o["slope"][ok]) * (8 + 2 * np.abs(ln_chi[ok]) + 8 * chi_cond) + 4 * np.abs(o["lnval"][ok]))
    bad = np.nonzero(rel > bound)[0]
    assert bad.size == 0, (rel[bad[:5]], bound[bad[:5]])
    assert np.all(d_gpu[~ok] <= 1.0000001 * d_orc[~ok])


# ----------------------------------------------------------------------------- Schwinger rate
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("n", [100003, 5, 1])
def test_schwinger_rate(orc, qed, ctx, dtype, n):
    """PAPER.md eqs.19-22 against the oracle's binary128 evaluation.  Tolerance on ln(rate): the rate is
    exp(-pi/eps) of the field invariants, so a rounding of the invariants F, G is amplified by (2 + pi/eps) kappa,
    kappa = d ln(eps^2) per unit relative rounding (order 1 for E parallel B, infinite for a plane wave)."""
    rng = np.random.default_rng(3)
    amp = np.exp(rng.uniform(np.log(0.02), np.log(2.0), n))
    e = [np.ascontiguousarray((amp * rng.normal(size=n)).astype(dtype)) for _ in range(3)]
    b = [np.ascontiguousarray((amp * rng.normal(size=n)).astype(dtype)) for _ in range(3)]
    if n > 100:  # special geometries: pure E, pure B, plane wave, E parallel B
        for k in range(3):
            b[k][0] = 0
            e[k][1] = 0
        e[0][2], e[1][2], e[2][2], b[0][2], b[1][2], b[2][2] = 0.3, 0, 0, 0, 0.3, 0
        e[0][3], e[1][3], e[2][3], b[0][3], b[1][3], b[2][3] = 0.4, 0, 0, 0.25, 0, 0
    got = ctx.schwinger_rate(to_dev(e), to_dev(b)).cpu().numpy()
    ref = orc.schwinger_rate(e, b)
    e64 = [np.asarray(a, np.float64) for a in e]
    b64 = [np.asarray(a, np.float64) for a in b]
    e2, b2 = sum(a * a for a in e64), sum(a * a for a in b64)
    F, G = 0.5 * (e2 - b2), sum(x * y for x, y in zip(e64, b64))
    root = np.sqrt(F * F + G * G)
    eps = np.sqrt(np.maximum(root + F, 1e-300))
    # conditioning of eps^2 = sqrt(F^2+G^2) + F with respect to roundings of F and G of size u (e^2 + b^2)
    rs = np.maximum(root, 1e-300)
    kappa = (e2 + b2) * (np.abs(1 + F / rs) + np.abs(G) / rs) / np.maximum(eps * eps, 1e-300)
    pos = ref > 1e-290
    assert np.all(got[~pos] <= 1e-280)
    err = np.abs(np.log(got[pos]) - np.log(ref[pos]))
    # 4e-13: the kernel carries ln(prefactor) = 130 in the exponent (so that weak fields do not underflow early):
    # a few roundings of size 130 * 2^-53
    bound = 4e-13 + 1e-15 * (2 + np.pi / eps[pos]) * kappa[pos]
    w = int(np.argmax(err / bound))
    assert np.all(err <= bound), (err[w], bound[w], eps[pos][w], kappa[pos][w], got[pos][w], ref[pos][w])
    if n > 100:
        assert got[1] == 0 and got[2] == 0 and got[0] > 0 and got[3] > 0
        assert np.median(err) < 2e-13
