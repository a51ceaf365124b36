"""GPU parity of the unit systems (picsarqed_set_units): the same physical particles
given in SI / normalised / Heaviside-Lorentz units must give what the oracle gives for the converted arrays, with the
momenta of parents and secondaries returned in the caller's units."""
import numpy as np
import pytest

from parity_common import LEPTON, PHOTON, assert_chi_close, check_evolve, code, to_dev, to_host

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def qed():
    import paper_2110_00256_b200 as q
    return q


@pytest.fixture(scope="module")
def mid_tables(orc):
    p = orc.TableParams(qs_chi_min=1e-3, qs_chi_max=1e3, qs_n_chi=40, qs_xi_min=1e-12, qs_n_xi=96,
                        bw_chi_min=2e-2, bw_chi_max=1e3, bw_n_chi=40, bw_n_xi=96)
    return orc.build_tables(p)


@pytest.fixture()
def ctx(qed, mid_tables):
    c = qed.Context(0)
    tp = mid_tables.params
    c.import_tables(qed.TableParams(**{k: getattr(tp, k) for k in tp.__dataclass_fields__}), mid_tables.lnG,
                    mid_tables.qs_lnP, mid_tables.lnT, mid_tables.bw_P)
    yield c
    c.close()


SYSTEMS = [(1, 0.0, "SI"), (2, 2.354564e15, "norm_omega"), (3, 0.8e-6, "norm_lambda"), (4, 0.0, "HL_MeV")]


def test_scales_agree_with_the_oracle(qed, ctx):
    from oracle import units as U
    for system, ref, _ in SYSTEMS:
        ctx.set_units(system, ref)
        assert np.allclose(ctx.unit_scales(), U.scales(system, ref), rtol=1e-14)
    ctx.set_units(0)
    assert ctx.unit_scales() == (1.0, 1.0, 1.0, 1.0)
    with pytest.raises(qed.PicsarQedError):
        ctx.set_units(2, 0.0)
    with pytest.raises(qed.PicsarQedError):
        ctx.set_units(9)


@pytest.mark.parametrize("system,ref,name", SYSTEMS)
@pytest.mark.parametrize("species", [LEPTON, PHOTON])
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_step_in_other_units(orc, qed, ctx, mid_tables, system, ref, name, species, dtype):
    """chi, evolve and the fused step on arrays in the caller's units.  The oracle works on the arrays converted with
    the library's own multipliers (pinned against the oracle's in test_scales_agree_with_the_oracle), so both sides
    see the same numbers and flags, counts and order must agree exactly."""
    import torch
    n = 30011
    pl, el, bl = qed.workloads.config1(seed=51, n=n, species=species, dtype=np.float64)
    ctx.set_units(system, ref)
    sp, se, sb, st = ctx.unit_scales()
    # the caller's arrays: library values divided by the multipliers, stored in the particle type
    pu = [np.ascontiguousarray((a / sp).astype(dtype)) for a in pl]
    eu = [np.ascontiguousarray((a / se).astype(dtype)) for a in el]
    bu = [np.ascontiguousarray((a / sb).astype(dtype)) for a in bl]
    # what both sides compute on: caller's value * multiplier, in fp64
    p = [a.astype(np.float64) * sp for a in pu]
    e = [a.astype(np.float64) * se for a in eu]
    b = [a.astype(np.float64) * sb for a in bu]
    tables = mid_tables.with_fp32_reads(dtype == np.float32)
    # chi
    out = torch.empty(n, dtype=torch.from_numpy(pu[0]).dtype, device="cuda")
    ctx.chi(species, to_dev(pu), to_dev(eu), to_dev(bu), out)
    ref_chi = orc.chi(species, p, e, b)
    assert_chi_close(out.cpu().numpy(), ref_chi, species, p, e, b)
    # fused step
    dt_lib = qed.workloads.choose_dt(orc.rate(tables, species, p, e, b), 0.15)
    dt_user = dt_lib / st
    tau0 = orc.init_optical_depth(species, code(dtype), n, 9).astype(dtype)
    dp, de, db = to_dev(pu), to_dev(eu), to_dev(bu)
    dtau = torch.from_numpy(tau0.copy()).cuda()
    nsec = 1 if species == LEPTON else 2
    tdt = dtau.dtype
    sec_p = [[torch.full((n,), -7.0, dtype=dp[0].dtype, device="cuda") for _ in range(3)] for _ in range(nsec)]
    sec_tau = [torch.full((n,), -7.0, dtype=tdt, device="cuda") for _ in range(nsec)]
    parent = torch.full((n,), -1, dtype=torch.int64, device="cuda")
    n_out = torch.zeros(1, dtype=torch.int64, device="cuda")
    # evolve alone first (on a copy) for the tie protocol
    tau_mid_t = dtau.clone()
    ctx.evolve_optical_depth(species, dp, de, db, dt_user, tau_mid_t)
    tau_mid = tau_mid_t.cpu().numpy()
    o = orc.evolve_optical_depth(tables, species, code(dtype), p, e, b, dt_user * st, tau0)
    check_evolve(tau_mid, tau0.astype(np.float64), o, dtype, np.log(np.maximum(ref_chi, 1e-300)))
    ctx.qed_step(species, dp, de, db, dtau, dt_user, 9, 4, 1000, n, sec_p[0], sec_tau[0],
                 sec_p[1] if nsec == 2 else None, sec_tau[1] if nsec == 2 else None, parent, n_out)
    fired = ctx.read_count(n_out)
    ids = 1000 + np.arange(n, dtype=np.uint64)
    if species == LEPTON:
        oe = orc.generate_photons(tables, code(dtype), code(dtype), p, e, b, tau_mid, 9, 4, ids, n)
        osec = [oe["ph_p"]]
    else:
        oe = orc.generate_pairs(tables, code(dtype), code(dtype), p, e, b, tau_mid, 9, 4, ids, n)
        osec = [oe["el_p"], oe["po_p"]]
    assert fired == oe["n_fired"] and fired > 0.05 * n
    assert np.array_equal(parent.cpu().numpy()[:fired], oe["parent"])
    tol = 1e-9 if dtype == np.float64 else 1e-5
    # momenta come back in the caller's units
    got_parent = [t.cpu().numpy().astype(np.float64) * sp for t in dp]
    norm = np.sqrt(sum(a * a for a in p)) + 1e-300
    for c in range(3):
        assert np.all(np.abs(got_parent[c] - oe["p"][c]) <= tol * norm)
    for s_ in range(nsec):
        g = [t.cpu().numpy().astype(np.float64)[:fired] * sp for t in sec_p[s_]]
        nrm = np.sqrt(sum(a * a for a in osec[s_])) + 1e-300
        for c in range(3):
            assert np.all(np.abs(g[c] - osec[s_][c]) <= tol * nrm), (s_, c)
            assert bool((sec_p[s_][c][fired:] == -7.0).all())
    assert np.array_equal(dtau.cpu().numpy() < 0, oe["tau"] < 0)


def test_closed_loop_calls_refuse_other_units(qed, ctx):
    import torch
    ctx.set_units(1)
    p = [torch.ones(8, dtype=torch.float64, device="cuda") for _ in range(3)]
    with pytest.raises(qed.PicsarQedError):
        ctx.boris_push_uniform(p, -1, (0, 0, 0), (0, 0, 1e-3), 1e-18)
    ctx.set_units(0)
    ctx.boris_push_uniform(p, -1, (0, 0, 0), (0, 0, 1e-3), 1e-18)
