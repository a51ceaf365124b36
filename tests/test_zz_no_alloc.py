"""picsarqed_generate_photons_noalloc (include/picsarqed.h): generate_photons on the library's static device scratch,
for callers that must not allocate.  Checked against the existing picsarqed_generate_photons on identical inputs: the
same kernels run on the same data, so everything is compared bit for bit -- on calls in a row that share the static
array (a large call, then a small one that finds the large one's counts, offsets and sums in it, then the large one
again), all dtype pairs, with a capacity cut, plus the size limit and the empty call.

Collected last on purpose (the suite runs with pytest -x).  Needs nothing from the other test files: its own context,
GPU-built tables, seeded inputs.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

DTYPES = [(np.float64, np.float64), (np.float32, np.float32), (np.float32, np.float64)]
IDS = ["f64", "f32", "f32_tau64"]


@pytest.fixture(scope="module")
def qed():
    import paper_2110_00256_b200 as q
    return q


@pytest.fixture(scope="module")
def ctx(qed):
    c = qed.Context(0)
    c.build_tables(qed.TableParams(qs_n_chi=64, qs_n_xi=96, bw_n_chi=64, bw_n_xi=96))
    yield c
    c.close()


def _inputs(qed, seed, n, dtype, tdtype, fired_fraction):
    import torch
    p, e, b = qed.workloads.config1(seed=seed, n=n, species=qed.LEPTON, dtype=dtype)
    rng = np.random.default_rng(1000 + seed)
    tau = rng.exponential(size=n).astype(tdtype)
    fired = rng.uniform(size=n) < fired_fraction
    fired[:40] = True        # a dense run: a chunk with more events than a staged segment would hold
    fired[-1] = True         # the ragged end
    if n > 3 * 4096:
        fired[4096:2 * 4096] = False   # an empty tile
    tau[fired] *= -1
    dev = lambda arrs: [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrs]
    return dev(p), dev(e), dev(b), torch.from_numpy(tau).cuda(), int(fired.sum())


def _run(call, p, e, b, tau, seed, step, id_base, capacity):
    """one call on copies of the inputs; returns everything it wrote"""
    import torch
    p = [t.clone() for t in p]
    tau = tau.clone()
    m = max(capacity, 1)
    ph_p = [torch.full((m,), -7.0, dtype=p[0].dtype, device="cuda") for _ in range(3)]
    ph_tau = torch.full((m,), -7.0, dtype=tau.dtype, device="cuda")
    parent = torch.full((m,), -1, dtype=torch.int64, device="cuda")
    n_out = torch.full((1,), -1, dtype=torch.int64, device="cuda")
    call(p, e, b, tau, seed, step, id_base, capacity, ph_p, ph_tau, parent, n_out)
    torch.cuda.synchronize()
    return dict(p=p, tau=tau, ph_p=ph_p, ph_tau=ph_tau, parent=parent, n_out=n_out)


def _assert_same(got, ref):
    import torch
    assert torch.equal(got["n_out"], ref["n_out"])
    assert torch.equal(got["parent"], ref["parent"])
    for k in ("p", "ph_p"):
        for a, r in zip(got[k], ref[k]):
            assert torch.equal(a, r), k
    # bit for bit, +inf and all (torch.equal treats equal infinities as equal; there are no NaNs here)
    assert torch.equal(got["tau"], ref["tau"]) and torch.equal(got["ph_tau"], ref["ph_tau"])


@pytest.mark.parametrize("dtype,tdtype", DTYPES, ids=IDS)
def test_noalloc_matches_generate_photons_on_calls_in_a_row(qed, ctx, dtype, tdtype):
    big = _inputs(qed, 11, 5 * 4096 * 8 + 1234, dtype, tdtype, 0.07)     # several tiles of 32 chunks, ragged end
    small = _inputs(qed, 12, 4096 + 77, dtype, tdtype, 0.3)              # fewer chunks than the call before it left behind
    calls = [(big, 21, 3, 1 << 33, None), (small, 22, 4, 5, None), (big, 23, 5, 0, None), (small, 24, 6, 9, 100)]
    for (p, e, b, tau, n_fired), seed, step, id_base, cap in calls:
        capacity = tau.numel() if cap is None else cap
        ref = _run(ctx.generate_photons, p, e, b, tau, seed, step, id_base, capacity)
        assert int(ref["n_out"].item()) == n_fired
        got = _run(ctx.generate_photons_noalloc, p, e, b, tau, seed, step, id_base, capacity)
        _assert_same(got, ref)
        # and again, straight after itself: the scratch now holds this very call's leftovers
        _assert_same(_run(ctx.generate_photons_noalloc, p, e, b, tau, seed, step, id_base, capacity), ref)


def test_noalloc_nothing_fires_and_empty(qed, ctx):
    import torch
    p, e, b, tau, _ = _inputs(qed, 13, 4096 * 3, np.float64, np.float64, 0.2)
    tau = tau.abs()
    got = _run(ctx.generate_photons_noalloc, p, e, b, tau, 1, 0, 0, tau.numel())
    assert int(got["n_out"].item()) == 0 and torch.equal(got["tau"], tau) and bool((got["parent"] == -1).all())
    z = torch.empty(0, dtype=torch.float64, device="cuda")
    n_out = torch.full((1,), -1, dtype=torch.int64, device="cuda")
    ctx.generate_photons_noalloc([z] * 3, [z] * 3, [z] * 3, z, 1, 0, 0, 0, [z] * 3, z, None, n_out)
    assert ctx.read_count(n_out) == 0


def test_noalloc_rejects_sizes_beyond_the_static_scratch(qed, ctx):
    """n > PICSARQED_NOALLOC_MAX_N: a clear error and nothing enqueued (the arrays are fp32 tau only: 64 MiB + 4 bytes)"""
    import torch
    n = qed.NOALLOC_MAX_N + 1
    tau = torch.ones(n, dtype=torch.float32, device="cuda")
    n_out = torch.full((1,), -1, dtype=torch.int64, device="cuda")
    arr = [tau] * 3
    with pytest.raises(qed.PicsarQedError, match="exceeds the static scratch"):
        ctx.generate_photons_noalloc(arr, arr, arr, tau, 1, 0, 0, 0, arr, tau, None, n_out)
    torch.cuda.synchronize()
    assert int(n_out.item()) == -1
    # the limit itself is served
    tau = tau[:qed.NOALLOC_MAX_N]
    arr = [tau] * 3
    ctx.generate_photons_noalloc(arr, arr, arr, tau, 1, 0, 0, 0, arr, tau, None, n_out)
    assert ctx.read_count(n_out) == 0
