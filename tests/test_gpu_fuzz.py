"""Randomised self-consistency of the three ways to take a step (SURVEY.md 8(c) P6 edge cases): picsarqed_qed_step,
picsarqed_evolve_optical_depth + picsarqed_generate_*, and picsarqed_step_host with a random number of slabs must
agree bit for bit -- counts, parent lists, order, momenta, optical depths, the capacity rule -- for sizes around every
tile and chunk border, every dtype combination, firing fractions from 0 to 0.9 and capacities from 1 to n + 5.
(Each path is held to the oracle by test_gpu_parity.py; this test sweeps the corners those cases do not enumerate.)"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def dev(a):
    import torch
    return [torch.from_numpy(np.ascontiguousarray(x)).cuda() for x in a]


def test_three_paths_agree_on_random_corners():
    import torch
    import paper_2110_00256_b200 as q
    from paper_2110_00256_b200 import workloads as w
    ctx = q.Context(0)
    ctx.build_tables(q.TableParams(qs_n_chi=64, qs_n_xi=64, bw_n_chi=64, bw_n_xi=64))
    rng = np.random.default_rng(12345)
    for trial in range(150):
        species = int(rng.integers(0, 2))
        dtype, tdtype = [(np.float64, np.float64), (np.float32, np.float32), (np.float32, np.float64)][int(rng.integers(0, 3))]
        n = int(rng.choice([1, 2, 3, 31, 32, 33, 127, 128, 129, 255, 1023, 1024, 1025, 2047, 2048, 2049, 3071, 4095, 4096, 4097, 8191, 12289, int(rng.integers(1, 40000))]))
        target = float(rng.choice([0.0, 0.01, 0.05, 0.3, 0.9]))
        p, e, b = w.config1(seed=int(rng.integers(1, 1 << 30)), n=n, species=species, dtype=dtype)
        pdt = torch.float64 if dtype == np.float64 else torch.float32
        tdt = torch.float64 if tdtype == np.float64 else torch.float32
        tau0 = torch.empty(n, dtype=tdt, device='cuda'); ctx.init_optical_depth(species, tau0, trial, 7)
        # dt from rates
        probe = torch.zeros(n, dtype=tdt, device='cuda')
        ctx.evolve_optical_depth(species, dev(p), dev(e), dev(b), 1.0, probe)
        rates = (-probe).double().cpu().numpy()
        dt = w.choose_dt(rates, target) if target > 0 and rates.max() > 0 else 0.0
        cap = int(rng.choice([n, max(1, n // 3), 1, n + 5]))
        nsec = 1 if species == 0 else 2
        def bufs():
            return ([[torch.full((cap,), -7.0, dtype=pdt, device='cuda') for _ in range(3)] for _ in range(nsec)],
                    [torch.full((cap,), -7.0, dtype=tdt, device='cuda') for _ in range(nsec)],
                    torch.full((cap,), -1, dtype=torch.int64, device='cuda'), torch.zeros(1, dtype=torch.int64, device='cuda'))
        # fused
        dp, de, db = dev(p), dev(e), dev(b); t1 = tau0.clone(); s1, st1, par1, c1 = bufs()
        ctx.qed_step(species, dp, de, db, t1, dt, 3, trial, 11, cap, s1[0], st1[0], s1[1] if nsec == 2 else None, st1[1] if nsec == 2 else None, par1, c1)
        # unfused
        dp2, t2 = dev(p), tau0.clone(); s2, st2, par2, c2 = bufs()
        ctx.evolve_optical_depth(species, dp2, de, db, dt, t2)
        if species == 0: ctx.generate_photons(dp2, de, db, t2, 3, trial, 11, cap, s2[0], st2[0], par2, c2)
        else: ctx.generate_pairs(dp2, de, db, t2, 3, trial, 11, cap, s2[0], st2[0], s2[1], st2[1], par2, c2)
        # host path with random slabs
        ctx.set_option("host_slabs", int(rng.choice([0, 1, 2, 5])))
        hp = [torch.from_numpy(np.ascontiguousarray(x)).pin_memory() for x in p]
        he = [torch.from_numpy(np.ascontiguousarray(x)).pin_memory() for x in e]; hb = [torch.from_numpy(np.ascontiguousarray(x)).pin_memory() for x in b]
        ht = tau0.cpu().pin_memory()
        hs = [torch.full((cap,), -7.0, dtype=tdt if k % 4 == 3 else pdt).pin_memory() for k in range(4 * nsec)]
        hpar = torch.full((cap,), -1, dtype=torch.int64).pin_memory()
        fired_h = ctx.step_host(species, hp, he, hb, ht, dt, 3, trial, 11, cap, hs, hpar)
        f1, f2 = ctx.read_count(c1), ctx.read_count(c2)
        eq = lambda a, b_: torch.equal(a, b_) or bool(((a == b_) | (a.isnan() & b_.isnan())).all())
        ok = f1 == f2 == fired_h and eq(t1, t2) and eq(t1.cpu(), ht) and eq(par1, par2) and eq(par1.cpu(), hpar)
        for k in range(3): ok = ok and eq(dp[k], dp2[k]) and eq(dp[k].cpu(), hp[k])
        for s_ in range(nsec):
            ok = ok and eq(st1[s_], st2[s_]) and eq(st1[s_].cpu(), hs[4 * s_ + 3])
            for k in range(3): ok = ok and eq(s1[s_][k], s2[s_][k]) and eq(s1[s_][k].cpu(), hs[4 * s_ + k])
        m = min(f1, cap)
        ok = ok and bool((par1[m:] == -1).all()) and (m == 0 or bool((par1[:m][1:] > par1[:m][:-1]).all()))
        neg = int((t1 < 0).sum().item())
        ok = ok and neg == max(0, f1 - cap)
        assert ok, ("trial", trial, species, dtype.__name__, tdtype.__name__, n, target, cap, f1, f2, fired_h)
    ctx.close()
