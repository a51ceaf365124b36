"""GPU table builder (picsarqed_build_tables) against the oracle's quadrature (BASELINE config 4:
"compare with the oracle quadrature at 1e-8 relative error").  Tolerances:
|d lnG|, |d lnT|, |d lnP_QS| <= 1e-8 absolute (= relative on G, T, P); |d P_BW| <= 1e-8 P + 1e-300."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-8


@pytest.fixture(scope="module")
def qed():
    import paper_2110_00256_b200 as q
    return q


def _chi_grid(lo, hi, n):
    return np.exp(np.log(lo) + (np.log(hi) - np.log(lo)) * np.arange(n) / (n - 1))


def _check_rows(orc, qed, ctx, kw, rows_qs, rows_bw, one_d_idx):
    op = orc.TableParams(**kw)
    lnG, lnT = ctx.export_tables(qed.TAB_LNG), ctx.export_tables(qed.TAB_LNT)
    qs, bw = ctx.export_tables(qed.TAB_QS_LNP), ctx.export_tables(qed.TAB_BW_P)
    # invariants at full size
    assert np.all(np.isfinite(lnG)) and np.all(np.isfinite(lnT)) and not np.isnan(qs).any() and not np.isnan(bw).any()
    assert np.all(np.diff(qs, axis=1) >= 0) and np.all(np.diff(bw, axis=1) >= 0)        # rows non-decreasing
    assert np.all(qs[:, -1] == 0.0) and np.all(bw[:, -1] == 0.5) and np.all(bw[:, 0] == 0.0)
    assert np.all(qs <= 0) and np.all(bw >= 0)
    assert np.all(np.diff(lnG) > 0)                                                     # G grows with chi
    # element-by-element against the oracle, on sampled rows (the oracle needs ~1 s per row)
    for r in rows_bw:
        ref = orc.build_bw_rows(op, r, r + 1)[0]
        assert np.all(np.abs(bw[r] - ref) <= TOL * ref + 1e-300), ("bw row", r)
    same_grid = op.rows_2d()[0] == op.qs_n_chi
    for r in rows_qs:
        ref, tot = orc.build_qs_rows(op, r, r + 1, return_total=True)
        assert np.all(np.abs(qs[r] - ref[0]) <= TOL), ("qs row", r)
        if same_grid:
            assert abs(lnG[r] - np.log(tot[0])) <= TOL
    chi_bw = _chi_grid(kw["bw_chi_min"], kw["bw_chi_max"], kw["bw_n_chi"])
    chi_qs = _chi_grid(kw["qs_chi_min"], kw["qs_chi_max"], kw["qs_n_chi"])
    for i in one_d_idx:
        ib, iq = min(i, chi_bw.size - 1), min(i, chi_qs.size - 1)
        assert abs(lnT[ib] - orc.bw_lnT(chi_bw[ib])) <= TOL
        assert abs(lnG[iq] - np.log(orc.qs_G(chi_qs[iq]))) <= TOL
    return lnG, lnT, qs, bw


def test_small_tables_full(orc, qed):
    """every entry of a small table set (C1 ranges)"""
    kw = dict(qs_chi_min=1e-3, qs_chi_max=1e3, qs_n_chi=24, qs_xi_min=1e-12, qs_n_xi=40,
              bw_chi_min=2e-2, bw_chi_max=1e3, bw_n_chi=24, bw_n_xi=40)
    ctx = qed.Context(0)
    ctx.build_tables(qed.TableParams(**kw))
    _check_rows(orc, qed, ctx, kw, range(24), range(24), range(24))
    ctx.close()


def test_coarse_and_odd_geometries(orc, qed):
    """coarse grids (wide cells: many panels per cell), a large xi_min, tiny row counts"""
    kw = dict(qs_chi_min=1e-4, qs_chi_max=1e3, qs_n_chi=5, qs_xi_min=1e-3, qs_n_xi=7,
              bw_chi_min=1e-3, bw_chi_max=5e3, bw_n_chi=6, bw_n_xi=3)
    ctx = qed.Context(0)
    ctx.build_tables(qed.TableParams(**kw))
    _check_rows(orc, qed, ctx, kw, range(5), range(6), range(6))
    kw = dict(qs_chi_min=0.5, qs_chi_max=2.0, qs_n_chi=2, qs_xi_min=0.2, qs_n_xi=2,
              bw_chi_min=0.5, bw_chi_max=2.0, bw_n_chi=2, bw_n_xi=2)
    ctx.build_tables(qed.TableParams(**kw))
    _check_rows(orc, qed, ctx, kw, range(2), range(2), range(2))
    ctx.close()


def test_config1_tables(orc, qed):
    kw = qed.workloads.table_params(1)
    ctx = qed.Context(0)
    ctx.build_tables(qed.TableParams(**kw))
    _check_rows(orc, qed, ctx, kw, [0, 37, 128, 255], [0, 41, 130, 255], [0, 1, 100, 254, 255])
    ctx.close()


def test_config4_tables(orc, qed):
    """BASELINE config 4: 4096-point ln G / ln T on [1e-4, 1e3] and 2048 x 2048 CDF tables (their own row grid): every
    64th row of both 2D tables (and the last) and every 64th 1D node (and the last) against the oracle quadrature"""
    kw = qed.workloads.table_params(4)
    ctx = qed.Context(0)
    ctx.build_tables(qed.TableParams(**kw))
    assert ctx.export_tables(qed.TAB_QS_LNP).shape == (2048, 2048) and ctx.export_tables(qed.TAB_LNG).shape == (4096,)
    rows = list(range(0, 2048, 64)) + [2047]
    nodes = list(range(0, 4096, 64)) + [1, 4094, 4095]
    lnG, lnT, qs, bw = _check_rows(orc, qed, ctx, kw, rows, rows, nodes)
    # pins of the paper/mathematics on the GPU tables themselves: T e^{8/(3 chi)} -> 3 sqrt3/(16 sqrt2) (chi -> 0),
    # G/chi -> 5 sqrt3/4 (chi -> 0)  [SURVEY.md 8(c) P3]
    assert abs(np.exp(lnT[0] + 8 / (3 * 1e-4)) / 0.2296396634 - 1) < 2e-4
    assert abs(np.exp(lnG[0]) / 1e-4 / 2.1650635095 - 1) < 2e-4
    ctx.close()


def test_own_row_grid_matches_shared_grid(qed):
    """a 2D table with its own row count holds the rows a table built on that grid alone would hold, bit for bit, and
    the 1D values are those of the 1D grid"""
    base = dict(qs_chi_min=1e-3, qs_chi_max=1e3, qs_xi_min=1e-9, qs_n_xi=33, bw_chi_min=2e-2, bw_chi_max=1e3, bw_n_xi=29)
    ctx = qed.Context(0)
    ctx.build_tables(qed.TableParams(qs_n_chi=21, bw_n_chi=17, qs_n_chi_2d=9, bw_n_chi_2d=11, **base))
    mixed = [ctx.export_tables(k) for k in range(4)]
    ctx.build_tables(qed.TableParams(qs_n_chi=21, bw_n_chi=17, **base))
    one_d = [ctx.export_tables(k) for k in range(4)]
    ctx.build_tables(qed.TableParams(qs_n_chi=9, bw_n_chi=11, **base))
    two_d = [ctx.export_tables(k) for k in range(4)]
    assert mixed[1].shape == (9, 33) and mixed[3].shape == (11, 29)
    # (1D values alone are integrated over at most 64 wide cells: the same integral, other panel ends)
    assert np.allclose(mixed[0], one_d[0], rtol=0, atol=1e-11) and np.allclose(mixed[2], one_d[2], rtol=0, atol=1e-11)
    assert np.array_equal(mixed[1], two_d[1]) and np.array_equal(mixed[3], two_d[3])
    ctx.close()


def test_import_export_roundtrip_and_errors(qed):
    kw = dict(qs_chi_min=1e-3, qs_chi_max=1e3, qs_n_chi=4, qs_xi_min=1e-6, qs_n_xi=5,
              bw_chi_min=1e-2, bw_chi_max=1e3, bw_n_chi=3, bw_n_xi=6)
    tp = qed.TableParams(**kw)
    rng = np.random.default_rng(0)
    t = [rng.normal(size=n) for n in tp.sizes()]
    ctx = qed.Context(0)
    with pytest.raises(qed.PicsarQedError):   # no tables yet
        import torch
        z = [torch.zeros(4, dtype=torch.float64, device="cuda") for _ in range(3)]
        ctx.evolve_optical_depth(0, z, z, z, 1e-15, torch.ones(4, dtype=torch.float64, device="cuda"))
    ctx.import_tables(tp, *t)
    for which in range(4):
        assert np.array_equal(ctx.export_tables(which).ravel(), t[which])
    with pytest.raises(qed.PicsarQedError):
        ctx.build_tables(qed.TableParams(**dict(kw, qs_chi_min=-1.0)))
    ctx.close()
