#!/usr/bin/env python
"""QED Monte Carlo step throughput on B200 (BASELINE.json metric, configuration 2 at N = 1).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--particles n]

A "step" is one pass of the whole hot path over the population: the fused chi + table lookup +
optical-depth kernel over all particles, then event generation (inverse-CDF sampling, secondaries
compacted in parent order, optical depth re-drawn).  Workload: 16 Mi electrons, fp64, gamma
log-uniform on [1e2, 1e5], fields re-drawn every step so that chi is log-uniform on ~[1e-3, 1e2],
1024-point ln G table and 1024x1024 photon-energy CDF table built on the GPU, dt such that ~5 % of
the particles fire per step.  Prints ONE JSON line (contract in DESIGN.md "Bench").
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "QED MC step particles/sec (fp64/fp32) at 1 B200; achieved HBM GB/s vs peak"
UNIT = "particles/s"
SEED = 2
BYTES_PER_PARTICLE_EVOLVE = 88  # 9 reads + tau read + tau write, fp64
# dram__bytes_read.sum + dram__bytes_write.sum of one launch of the evolve pass at 16 Mi particles, from the ncu --set full
# capture named in EVOLVE_TRAFFIC_SOURCE (1.3436 GB read = the 80 B/particle of inputs; 109 MB written: part of the 134 MB
# of new tau is still dirty in L2 when the kernel ends, plus the staged records).  A profile figure, not a measurement of
# the timed run: the line says so in `traffic_source`, and carries it only at the profiled size.
EVOLVE_TRAFFIC_SOURCE = "profiles/r2_step_full.md (ncu --set full, dram__bytes_read.sum + dram__bytes_write.sum, 16 Mi particles)"
EVOLVE_DRAM_TRAFFIC_BYTES = 1343574000 + 109243392


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--particles", type=int, default=1 << 24, help="particles per GPU (default 16 Mi = config 2)")
    ap.add_argument("--field-sets", type=int, default=4, help="distinct per-step field sets kept in HBM")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--cpu-sample", type=int, default=1 << 23, help="particles in the oracle timing sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true",
                    help="only the headline configuration 2 (skip configs 3, 5 and 4 in `other_configs`)")
    ap.add_argument("--dt-scale", type=float, default=1.0, help="multiply the 5 %% time step (tuning experiments)")
    ap.add_argument("--opt", action="append", default=[], metavar="NAME=VALUE",
                    help="picsarqed_set_option before the run (tuning experiments), e.g. --opt fused_step=0")
    ap.add_argument("--cascade", action="store_true",
                    help="secondary workload (SURVEY.md 8(f)-1): closed loop of Ridgers case (iii) instead of the "
                         "headline step; prints its own JSON line")
    ap.add_argument("--cascade-dtype", default="f64", choices=["f64", "f32"])
    ap.add_argument("--tables", action="store_true",
                    help="secondary workload (BASELINE config 4): build the 4096-point 1D tables and the 4096x2048 2D "
                         "tables on the GPU; prints its own JSON line")
    return ap.parse_args()


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0}, "fallback"


class ClockSampler(threading.Thread):
    """samples SM clock and throttle reasons through NVML while the timed region runs"""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.stop_flag, self.max_mhz = index, [], set(), False, None

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            names = {"sw_power_cap": nv.nvmlClocksEventReasonSwPowerCap, "hw_slowdown": nv.nvmlClocksEventReasonHwSlowdown,
                     "hw_thermal_slowdown": nv.nvmlClocksEventReasonHwThermalSlowdown,
                     "sw_thermal_slowdown": nv.nvmlClocksEventReasonSwThermalSlowdown}
            while not self.stop_flag:
                self.samples.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksEventReasons(h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
                time.sleep(0.002)
        except Exception as exc:  # NVML missing: report it, do not hide it
            self.reasons.add("nvml_unavailable: %s" % type(exc).__name__)

    def summary(self):
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------------------------------------
#  the oracle, timed on the host cores (cpu_baseline leg and --impl reference)
# ------------------------------------------------------------------------------------------------
def oracle_tables_from(tp_kwargs, tables):
    import oracle
    return oracle.Tables(oracle.TableParams(**tp_kwargs), *tables)


def time_oracle(tp_kwargs, tables, n_sample, steps, dt, seed=SEED):
    """oracle evolve + generate_photons on the first n_sample particles of the workload; returns
    (particles/s, seconds, threads)"""
    import oracle
    from paper_2110_00256_b200 import workloads as w
    tabs = oracle_tables_from(tp_kwargs, tables)
    p, gamma = w.config2(seed=seed, n=n_sample)
    tau = oracle.init_optical_depth(0, 1, n_sample, seed)
    fields = [w.config2_fields(seed, s, gamma) for s in range(steps)]
    t0 = time.perf_counter()
    for s in range(steps):
        e, b = fields[s]
        tau = oracle.evolve_optical_depth(tabs, 0, 1, p, e, b, dt, tau)["tau"]
        o = oracle.generate_photons(tabs, 1, 1, p, e, b, tau, seed, s, capacity=n_sample // 8)
        p, tau = o["p"], o["tau"]
    sec = time.perf_counter() - t0
    return n_sample * steps / sec, sec, oracle.num_threads()


def reference_tables(tp_kwargs):
    """tables for the stand-alone reference arm: the oracle's own quadrature on a reduced grid would change the
    workload, and the full 1024x1024 oracle build takes ~10 core-minutes; the arm times the runtime path only,
    so it reads power-law stand-in tables of the right shape (values do not change the oracle's work per particle)."""
    n1, n2 = tp_kwargs["qs_n_chi"], tp_kwargs["qs_n_xi"]
    chi = np.exp(np.linspace(np.log(tp_kwargs["qs_chi_min"]), np.log(tp_kwargs["qs_chi_max"]), n1))
    lnG = np.log(2.165 * chi / (1 + chi) ** (1 / 3))
    lxi = np.log(tp_kwargs["qs_xi_min"]) * (1 - np.arange(n2) / (n2 - 1))
    qs = np.tile(lxi / 3, (n1, 1))
    m1, m2 = tp_kwargs["bw_n_chi"], tp_kwargs["bw_n_xi"]
    return lnG, qs, np.full(m1, -3.0), np.tile(np.linspace(0, 0.5, m2), (m1, 1))


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2110_00256_b200 import workloads as w
    tp = w.table_params(2)
    tables = reference_tables(tp)
    import oracle
    n = min(args.cpu_sample, args.particles)
    steps = max(1, args.steps)
    p0, g0 = w.config2(seed=SEED, n=1 << 16)
    e0, b0 = w.config2_fields(SEED, 0, g0)
    dt = w.choose_dt(oracle.rate(oracle_tables_from(tp, tables), 0, p0, e0, b0), 0.05)  # the 5 % rule
    for _ in range(max(0, min(args.warmup, 1))):
        time_oracle(tp, tables, min(n, 1 << 16), 1, dt)
    # bound the run: the oracle does ~4e6 particle-steps/s on 16 cores; the arm honours --particles (through --cpu-sample)
    # and --steps up to a wall-time cap, and says what it ran
    wall_cap_s = 60.0
    probe_n = min(n, 1 << 20)
    _, probe_sec, _ = time_oracle(tp, tables, probe_n, 1, dt)
    per_step = probe_sec * n / probe_n
    steps_run = int(max(1, min(steps, wall_cap_s // max(per_step, 1e-9))))
    value, sec, threads = time_oracle(tp, tables, n, steps_run, dt)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": steps_run,
            "warmup": args.warmup, "ms_per_step": 1e3 * sec / steps_run, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "config 2 (synchrotron emission, fp64), oracle on host cores", "particles": n,
                       "tables": "1024 / 1024x1024 (stand-in values, same shape)", "steps_asked": steps,
                       "steps_run": steps_run, "wall_cap_s": wall_cap_s},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle",
                             "sample": "%d particles x %d steps (evolve + photon emission)" % (n, steps_run)},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------
#  the other configurations of BASELINE.json (the fp32 half of the metric, the table build)
# ------------------------------------------------------------------------------------------------
def event_bytes(species, es, ts, with_parent_index):
    """algorithmic bytes of one event: the parent's momentum and optical depth rewritten, the
    secondaries (3 reals + optical depth each) written, 8 bytes of parent index when the caller asks for it"""
    nsec = 1 if species == 0 else 2
    return (3 * es + ts) + nsec * (3 * es + ts) + (8 if with_parent_index else 0)


def timed_steps(torch, ctx, step_fn, reseed_fn, steps, warmup):
    """per-step CUDA events on the context's stream; reseed_fn (restoring consumed photons) runs between steps, outside
    the timed brackets.  Returns (mean ms per step, evolve-pass ms, event-pass ms)"""
    for s in range(warmup):
        reseed_fn()
        step_fn(s)
    torch.cuda.synchronize()
    ctx.set_option("time_kernels", 1)
    ctx.get_timing()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for k in range(steps):
        reseed_fn()
        ev[k][0].record()
        step_fn(warmup + k)
        ev[k][1].record()
    torch.cuda.synchronize()
    ms_a, ms_b, calls = ctx.get_timing()
    ctx.set_option("time_kernels", 0)
    ms = float(np.mean([a.elapsed_time(b) for a, b in ev]))
    return ms, ms_a / max(steps, 1), ms_b / max(steps, 1)


def leg_roofline(peaks, peak_kind, kernel, evolve_bytes, ms_evolve, step_bytes, ms_step):
    ach = evolve_bytes / (ms_evolve * 1e-3) / 1e9
    whole = step_bytes / (ms_step * 1e-3) / 1e9
    return {"bound": "hbm", "kernel": kernel, "achieved": ach, "peak": peaks["hbm_gbs"],
            "peak_kind": peak_kind + " (MEASURED_PEAKS.json hbm_gbs, copy)", "unit": "GB/s", "frac": ach / peaks["hbm_gbs"],
            "traffic": None, "algorithmic_bytes_per_launch": evolve_bytes, "ms_per_launch": ms_evolve,
            "whole_step": {"algorithmic_bytes": step_bytes, "achieved": whole, "frac": whole / peaks["hbm_gbs"]}}


def run_config3(args, torch, q, w, ctx, dev, peaks, peak_kind):
    """BASELINE config 3: 16 Mi photons, fp32, Breit-Wheeler only; every event makes a pair; the photons that decayed are
    re-seeded between steps, so every step sees 16 Mi live photons"""
    n, seed = args.particles, 3
    cap = n // 8
    p_h, gamma = w.config3(seed=seed, n=n)
    n_sets = 4
    p = [torch.from_numpy(a).to(dev) for a in p_h]
    fields = []
    for s_ in range(n_sets):
        e_h, b_h = w.config3_fields(seed, s_, gamma)
        fields.append([torch.from_numpy(a).to(dev) for a in (*e_h, *b_h)])
    tau = torch.empty(n, dtype=torch.float32, device=dev)
    ctx.init_optical_depth(q.PHOTON, tau, seed, 0)
    p0, tau0 = [t.clone() for t in p], tau.clone()
    m = min(n, 1 << 16)
    probe = torch.zeros(m, dtype=torch.float32, device=dev)
    ctx.evolve_optical_depth(q.PHOTON, [t[:m] for t in p], [t[:m] for t in fields[0][:3]], [t[:m] for t in fields[0][3:]], 1.0, probe)
    dt = w.choose_dt((-probe).double().cpu().numpy(), 0.05)
    el = [torch.empty(cap, dtype=torch.float32, device=dev) for _ in range(4)]
    po = [torch.empty(cap, dtype=torch.float32, device=dev) for _ in range(4)]
    parent = torch.empty(cap, dtype=torch.int64, device=dev)
    n_out = torch.zeros(1, dtype=torch.int64, device=dev)

    def reseed():     # dead photons (p = 0, tau = +inf) come back as they were; the survivors keep their optical depth
        dead = torch.isinf(tau)
        for a, a0 in zip(p, p0):
            torch.where(dead, a0, a, out=a)
        torch.where(dead, tau0, tau, out=tau)

    def step(s_):
        f = fields[s_ % n_sets]
        ctx.qed_step(q.PHOTON, p, f[:3], f[3:], tau, dt, seed, s_, 0, cap, el[:3], el[3], po[:3], po[3], parent, n_out)

    steps = max(20, args.steps) if args.steps >= 5 else args.steps
    ms, ms_ev, ms_evt = timed_steps(torch, ctx, step, reseed, steps, args.warmup)
    fired = ctx.read_count(n_out)
    evolve_bytes = 44 * n
    step_bytes = evolve_bytes + event_bytes(1, 4, 4, True) * fired
    leg = {"workload": "config 3: Breit-Wheeler pair production only, fp32, %d photons, 1024-pt lnT + 1024x1024 pair CDF "
                       "(fp32 copy), evolve + pair creation per step, decayed photons re-seeded between steps" % n,
           "dtype": "f32", "value": n / (ms * 1e-3), "unit": UNIT, "ms_per_step": ms, "steps": steps,
           "fired_fraction_last_step": fired / n, "dt_s": dt,
           "timing": "mean of per-step CUDA events; the re-seeding of decayed photons runs between the brackets",
           "kernels_ms": {"evolve_pass": ms_ev, "event_pass": ms_evt},
           "roofline": leg_roofline(peaks, peak_kind, "evolve_kernel<float,float,PHOTON,U=1,EMIT> (evolve pass of qed_step)",
                                    evolve_bytes, ms_ev, step_bytes, ms)}
    if not args.no_cpu_baseline:
        import oracle
        ns, steps_cpu = min(n, 1 << 21), 3
        tabs = oracle_tables_from(w.table_params(3), [ctx.export_tables(k) for k in range(4)]).with_fp32_reads(True)
        ph, ga = w.config3(seed=seed, n=ns)
        tau_h = oracle.init_optical_depth(1, 0, ns, seed)
        flds = [w.config3_fields(seed, s_, ga) for s_ in range(steps_cpu)]
        t0 = time.perf_counter()
        for s_ in range(steps_cpu):
            e_, b_ = flds[s_]
            t_ = oracle.evolve_optical_depth(tabs, 1, 0, ph, e_, b_, dt, tau_h)["tau"]
            oracle.generate_pairs(tabs, 0, 0, ph, e_, b_, t_, seed, s_, capacity=ns // 8)
        sec = time.perf_counter() - t0
        leg["cpu_baseline"] = {"value": ns * steps_cpu / sec, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                               "sample": "first %d photons of the workload x %d steps (evolve + pair creation), %.1f s" % (ns, steps_cpu, sec)}
    return leg


def run_config5(args, torch, q, w, ctx, dev, peaks, peak_kind):
    """BASELINE config 5: 256 Mi leptons + 64 Mi photons, fp32 with fp64 optical depth, plane wave + noise; both
    processes per step.  The population is generated on the host in slabs of 16 Mi (seed 5 + 1000 slab: the same
    distribution as one draw of the whole), in parallel threads."""
    from concurrent.futures import ThreadPoolExecutor
    scale = args.particles / float(1 << 24)             # --particles scales every configuration alike
    n_lep, n_pho = int((1 << 28) * scale), int((1 << 26) * scale)
    slab = min(1 << 24, n_pho)
    seed = 5
    pops = {}

    def gen(job):
        sp, k, m = job
        return sp, k, w.config5(seed=seed + 1000 * k + 500 * sp, n=m, species=sp)

    for sp, n_sp in ((q.LEPTON, n_lep), (q.PHOTON, n_pho)):
        pops[sp] = [torch.empty(n_sp, dtype=torch.float32, device=dev) for _ in range(9)]
    jobs = [(sp, k, min(slab, n_sp - k * slab)) for sp, n_sp in ((q.LEPTON, n_lep), (q.PHOTON, n_pho))
            for k in range((n_sp + slab - 1) // slab)]
    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
        for sp, k, (p_h, e_h, b_h) in ex.map(gen, jobs):
            for a, h in zip(pops[sp], (*p_h, *e_h, *b_h)):
                a[k * slab:k * slab + h.size].copy_(torch.from_numpy(h))
    tau = {sp: torch.empty(pops[sp][0].numel(), dtype=torch.float64, device=dev) for sp in pops}
    id_base = {q.LEPTON: 0, q.PHOTON: n_lep}
    dts = []
    for sp in pops:
        ctx.init_optical_depth(sp, tau[sp], seed, id_base[sp])
        m = min(pops[sp][0].numel(), 1 << 16)
        probe = torch.zeros(m, dtype=torch.float64, device=dev)
        ctx.evolve_optical_depth(sp, [t[:m] for t in pops[sp][:3]], [t[:m] for t in pops[sp][3:6]], [t[:m] for t in pops[sp][6:]], 1.0, probe)
        dts.append((-probe).cpu().numpy())
    dt = w.choose_dt(np.concatenate(dts), 0.05)        # one time step for both species (5 % rule over both)
    cap = {sp: pops[sp][0].numel() // 4 for sp in pops}
    sec = {sp: [[torch.empty(cap[sp], dtype=torch.float32, device=dev) for _ in range(3)] for _ in range(1 + sp)] for sp in pops}
    sec_t = {sp: [torch.empty(cap[sp], dtype=torch.float64, device=dev) for _ in range(1 + sp)] for sp in pops}
    n_out = {sp: torch.zeros(1, dtype=torch.int64, device=dev) for sp in pops}
    ph = pops[q.PHOTON]
    ph0, tau_ph0 = [t.clone() for t in ph[:3]], tau[q.PHOTON].clone()

    def reseed():
        dead = torch.isinf(tau[q.PHOTON])
        for a, a0 in zip(ph[:3], ph0):
            torch.where(dead, a0, a, out=a)
        torch.where(dead, tau_ph0, tau[q.PHOTON], out=tau[q.PHOTON])

    def step(s_):
        for sp in (q.LEPTON, q.PHOTON):
            a = pops[sp]
            ctx.qed_step(sp, a[:3], a[3:6], a[6:], tau[sp], dt, seed, s_, id_base[sp], cap[sp], sec[sp][0], sec_t[sp][0],
                         sec[sp][1] if sp == q.PHOTON else None, sec_t[sp][1] if sp == q.PHOTON else None, None, n_out[sp])

    steps = 10 if args.steps >= 5 else args.steps
    ms, ms_ev, ms_evt = timed_steps(torch, ctx, step, reseed, steps, min(args.warmup, 3))
    fired = {sp: ctx.read_count(n_out[sp]) for sp in pops}
    n = n_lep + n_pho
    evolve_bytes = 52 * n
    step_bytes = evolve_bytes + sum(event_bytes(sp, 4, 8, False) * fired[sp] for sp in pops)
    leg = {"workload": "config 5: laser-plasma-like population, fp32 particles with fp64 optical depth, %d leptons + %d "
                       "photons, plane wave a0 = 500 + noise, both processes, compaction and re-draw per step; decayed photons "
                       "re-seeded between steps" % (n_lep, n_pho),
           "dtype": "f32 (optical depth f64)", "value": n / (ms * 1e-3), "unit": UNIT, "ms_per_step": ms, "steps": steps,
           "fired_fraction_last_step": {"leptons": fired[q.LEPTON] / n_lep, "photons": fired[q.PHOTON] / n_pho}, "dt_s": dt,
           "timing": "mean of per-step CUDA events; the re-seeding of decayed photons runs between the brackets",
           "kernels_ms": {"evolve_passes": ms_ev, "event_passes": ms_evt},
           "roofline": leg_roofline(peaks, peak_kind, "evolve_kernel<float,double,*,U=1,EMIT> (the two evolve passes of the step)",
                                    evolve_bytes, ms_ev, step_bytes, ms)}
    if not args.no_cpu_baseline:
        import oracle
        tabs = oracle_tables_from(w.table_params(5), [ctx.export_tables(k) for k in range(4)]).with_fp32_reads(True)
        ns = {q.LEPTON: min(n_lep, 1 << 21), q.PHOTON: min(n_pho, 1 << 19)}
        data = {sp: w.config5(seed=seed + 500 * sp, n=ns[sp], species=sp) for sp in ns}
        taus = {sp: oracle.init_optical_depth(sp, 1, ns[sp], seed) for sp in ns}
        steps_cpu = 3
        t0 = time.perf_counter()
        for s_ in range(steps_cpu):
            for sp in ns:
                p_, e_, b_ = data[sp]
                t_ = oracle.evolve_optical_depth(tabs, sp, 1, p_, e_, b_, dt, taus[sp])["tau"]
                (oracle.generate_photons if sp == q.LEPTON else oracle.generate_pairs)(tabs, 0, 1, p_, e_, b_, t_, seed, s_)
        sec_cpu = time.perf_counter() - t0
        leg["cpu_baseline"] = {"value": sum(ns.values()) * steps_cpu / sec_cpu, "unit": UNIT, "cores": oracle.num_threads(),
                               "kind": "oracle", "sample": "%d leptons + %d photons of the same recipe x %d steps (both processes), "
                                                           "%.1f s" % (ns[q.LEPTON], ns[q.PHOTON], steps_cpu, sec_cpu)}
    return leg


# FP64 warp instructions (DFMA + DMUL + DADD + DSETP, counted on the source page) of one build of the configuration-4 tables,
# summed over the four table_rows_kernel launches, from the ncu capture named in TABLES_FP64_SOURCE.  A profile figure of
# that build of the library; the live part of the roofline entry is the duration (CUDA events inside the library).
TABLES_FP64_SOURCE = "profiles/r2_tables_full.md"
TABLES_FP64_WARP_INST = 5036057619


def run_config4(args, torch, q, w, peaks):
    """BASELINE config 4: 4096-point lnG, lnT on [1e-4, 1e3] and 2048 x 2048 CDF tables from the Bessel quadratures.
    The kernel is bound by the FP64 pipe: roofline = FP64 warp instructions / time against 148 SMs x 4 sub-partitions x
    16 lanes x 1 instruction per 2 cycles... reported as the fraction of cycles the pipe could have issued"""
    ctx = q.Context(0)
    tp = q.TableParams(**w.table_params(4))
    times, dev = [], []
    for _ in range(2 + 5):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        ctx.build_tables(tp)
        times.append(time.perf_counter() - t0)
        dev.append(ctx.table_build_ms())
    ms = 1e3 * float(np.median(times[2:]))          # the call: quadrature + fp32 copies + search guides + synchronisation
    ms_dev = float(np.median(dev[2:]))              # the quadrature kernels alone (CUDA events inside the library)
    cells = tp.rows_2d()[0] * tp.qs_n_xi + tp.rows_2d()[1] * tp.bw_n_xi
    leg = {"workload": "config 4: table generation, fp64: 4096-point lnG and lnT on [1e-4, 1e3], two 2048 x 2048 CDF tables",
           "dtype": "f64", "metric": "table build time", "value": ms, "unit": "ms", "higher_is_better": False,
           "builds_timed": 5, "cells": cells, "cells_per_s": cells / (ms * 1e-3), "quadrature_kernels_ms": ms_dev}
    sm_mhz = peaks.get("sm_max_mhz", 1965.0)
    if TABLES_FP64_WARP_INST:
        # an SM issues one FP64 warp instruction every 2 cycles per sub-partition (16 lanes each, 64 FMA per SM per cycle)
        peak = 148 * 4 * 0.5 * sm_mhz * 1e6
        ach = TABLES_FP64_WARP_INST / (ms_dev * 1e-3)
        leg["roofline"] = {"bound": "alu", "kernel": "table_rows_kernel<QS>, table_rows_kernel<BW>", "achieved": ach / 1e12,
                           "peak": peak / 1e12, "unit": "T warp-instructions/s (FP64 pipe)", "frac": ach / peak, "traffic": None,
                           "peak_kind": "derived: 148 SMs x 4 sub-partitions x 1 FP64 warp instruction per 2 cycles x %.0f MHz" % sm_mhz,
                           "instruction_count_source": TABLES_FP64_SOURCE}
    if not args.no_cpu_baseline:
        import oracle
        op = oracle.TableParams(**w.table_params(4))
        rows = [0, 512, 1024, 1536, 2047]
        t0 = time.perf_counter()
        for r in rows:
            oracle.build_qs_rows(op, r, r + 1)
            oracle.build_bw_rows(op, r, r + 1)
        sec = time.perf_counter() - t0
        est_ms = 1e3 * sec / len(rows) * 2048      # both tables: 2048 row pairs (the 1D tables add 4096 + 4096 totals)
        leg["cpu_baseline"] = {"value": est_ms, "unit": "ms", "cores": oracle.num_threads(), "kind": "oracle",
                               "sample": "rows %s of both 2D tables by the oracle's adaptive quadrature, %.1f s, scaled to 2048 "
                                         "rows per table" % (rows, sec)}
    ctx.close()
    return leg


# ------------------------------------------------------------------------------------------------
#  the CUDA path
# ------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist

    import paper_2110_00256_b200 as q
    from paper_2110_00256_b200 import sharding
    from paper_2110_00256_b200 import workloads as w

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)
    n = args.particles
    seed = SEED + 1000 * rank      # every rank owns an independent shard (weak scaling, no data-path collective)
    id_base, _ = sharding.shard_range(rank, world, world * n)   # contiguous global particle ids per rank
    cap = n // 8

    ctx = q.Context(local)
    for kv in args.opt:
        name, value = kv.split("=")
        ctx.set_option(name, int(value))
    tp_kwargs = w.table_params(2)
    t0 = time.perf_counter()
    ctx.build_tables(q.TableParams(**tp_kwargs))
    table_build_s = time.perf_counter() - t0

    # ---- inputs: generated on the host (pinned), resident in HBM before the timed region -----------
    p_h, gamma = w.config2(seed=seed, n=n)
    n_sets = max(1, min(args.field_sets, args.steps + args.warmup))
    p_pin = [torch.from_numpy(a).pin_memory() for a in p_h]
    field_pin = []
    for s in range(n_sets):
        e_h, b_h = w.config2_fields(seed, s, gamma)
        field_pin.append([torch.from_numpy(a).pin_memory() for a in (*e_h, *b_h)])
    p = [t.to(dev) for t in p_pin]
    fields = [[t.to(dev) for t in fs] for fs in field_pin]
    tau = torch.empty(n, dtype=torch.float64, device=dev)
    ctx.init_optical_depth(q.LEPTON, tau, seed, id_base)
    ph_p = [torch.empty(cap, dtype=torch.float64, device=dev) for _ in range(3)]
    ph_tau = torch.empty(cap, dtype=torch.float64, device=dev)
    ph_parent = torch.empty(cap, dtype=torch.int64, device=dev)
    n_out = torch.zeros(1, dtype=torch.int64, device=dev)

    # ---- dt by the 5 % rule, rates from the CUDA path itself (tau = 0, dt = 1 s  ->  tau = -rate) ----
    m = min(n, 1 << 16)
    probe = torch.zeros(m, dtype=torch.float64, device=dev)
    ctx.evolve_optical_depth(q.LEPTON, [t[:m] for t in p], [t[:m] for t in fields[0][:3]],
                             [t[:m] for t in fields[0][3:]], 1.0, probe)
    dt = w.choose_dt((-probe).cpu().numpy(), 0.05) * args.dt_scale

    def step(s):
        f = fields[s % n_sets]
        ctx.qed_step(q.LEPTON, p, f[:3], f[3:], tau, dt, seed, s, id_base, cap, ph_p, ph_tau, None, None, ph_parent, n_out)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for s in range(args.warmup):
        step(s)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    while not sampler.samples and not sampler.reasons and sampler.is_alive():
        time.sleep(0.001)          # NVML is up before the timed region starts
    ctx.set_option("time_kernels", 1)  # CUDA events around the evolve pass and the event pass, on this stream
    ctx.get_timing()
    start, stop = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    start.record()
    for k in range(args.steps):
        step(args.warmup + k)      # evolve_kernel<..., EMIT> + tile_scan_kernel + event_kernel
    stop.record()
    barrier()
    sampler.stop_flag = True
    sampler.join()
    ms_total = start.elapsed_time(stop)
    ms_evolve, ms_events, n_timed = ctx.get_timing()
    ctx.set_option("time_kernels", 0)
    ms_evolve /= max(n_timed, 1)
    ms_events /= max(n_timed, 1)
    fired_last = ctx.read_count(n_out)
    # the two-call path (evolve_optical_depth, then generate_photons) on the same state, for comparison
    split = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(5)]
    for k in range(5):
        s = args.warmup + args.steps + k
        f = fields[s % n_sets]
        split[k][0].record()
        ctx.evolve_optical_depth(q.LEPTON, p, f[:3], f[3:], dt, tau)
        split[k][1].record()
        ctx.generate_photons(p, f[:3], f[3:], tau, seed, s, id_base, cap, ph_p, ph_tau, ph_parent, n_out)
        split[k][2].record()
    barrier()
    ms_evolve2 = float(np.mean([e[0].elapsed_time(e[1]) for e in split[1:]]))
    ms_events2 = float(np.mean([e[1].elapsed_time(e[2]) for e in split[1:]]))
    # the same two calls with "stage_records" (the caller promises not to touch the arrays in between)
    ctx.set_option("stage_records", 1)
    for k in range(5):
        s = args.warmup + args.steps + 5 + k
        f = fields[s % n_sets]
        split[k][0].record()
        ctx.evolve_optical_depth(q.LEPTON, p, f[:3], f[3:], dt, tau)
        split[k][1].record()
        ctx.generate_photons(p, f[:3], f[3:], tau, seed, s, id_base, cap, ph_p, ph_tau, ph_parent, n_out)
        split[k][2].record()
    barrier()
    ctx.set_option("stage_records", 0)
    ms_evolve3 = float(np.mean([e[0].elapsed_time(e[1]) for e in split[1:]]))
    ms_events3 = float(np.mean([e[1].elapsed_time(e[2]) for e in split[1:]]))
    ms_total = sharding.max_over_ranks(ms_total, dev)
    value = world * n * args.steps / (ms_total * 1e-3)

    # ---- end to end through the C ABI with HOST buffers (copies inside the timed region) -------------
    tau_pin = tau.cpu().pin_memory()
    p_e2e = [t.clone().pin_memory() for t in p_pin]
    sec_pin = [torch.empty(cap, dtype=torch.float64).pin_memory() for _ in range(4)]
    ctx.step_host(q.LEPTON, p_e2e, field_pin[0][:3], field_pin[0][3:], tau_pin, dt, seed, 10_000, id_base, cap, sec_pin)
    barrier()
    t0 = time.perf_counter()
    fired_e2e = 0
    for k in range(args.e2e_steps):
        f = field_pin[k % n_sets]
        fired_e2e = ctx.step_host(q.LEPTON, p_e2e, f[:3], f[3:], tau_pin, dt, seed, 10_001 + k, id_base, cap, sec_pin)
    barrier()
    e2e_s = time.perf_counter() - t0
    e2e_s = sharding.max_over_ranks(e2e_s, dev)
    e2e_value = world * n * args.e2e_steps / e2e_s
    h2d = 10 * n * 8
    d2h = 4 * n * 8 + 8 + min(fired_e2e, cap) * 4 * 8

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    peaks, peak_kind = measured_peaks()
    # dominant kernel: the evolve pass (evolve_kernel<double,double,LEPTON,2,EMIT>): 88 algorithmic bytes per particle
    # (SURVEY.md 8(d)); the 48-byte records it stages for the ~5 % that fire are not counted as algorithmic
    evolve_bytes = BYTES_PER_PARTICLE_EVOLVE * n
    achieved = evolve_bytes / (ms_evolve * 1e-3) / 1e9
    step_bytes = evolve_bytes + event_bytes(0, 8, 8, True) * fired_last
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "config 2: synchrotron (nonlinear Compton) emission only, fp64, %d electrons per GPU, "
                               "1024-pt lnG + 1024x1024 photon CDF (GPU-built), evolve + photon emission per step" % n,
                   "particles_per_gpu": n, "dt_s": dt, "fired_fraction_last_step": fired_last / n,
                   "l2": "inputs larger than L2: %d field sets x %d MB cycled, %d MB of momenta/tau" % (
                       n_sets, 6 * n * 8 >> 20, 4 * n * 8 >> 20),
                   "parallelism": "independent shards per GPU" if world > 1 else "single GPU",
                   "table_build_s": table_build_s},
        "roofline": {"bound": "hbm", "kernel": "evolve_kernel<double,double,LEPTON,U=2,EMIT> (evolve pass of qed_step)",
                     "achieved": achieved,
                     "peak": peaks["hbm_gbs"], "peak_kind": peak_kind + " (MEASURED_PEAKS.json hbm_gbs, copy)",
                     "unit": "GB/s", "frac": achieved / peaks["hbm_gbs"],
                     "traffic": EVOLVE_DRAM_TRAFFIC_BYTES if n == 1 << 24 else None, "traffic_source": EVOLVE_TRAFFIC_SOURCE,
                     "algorithmic_bytes_per_launch": evolve_bytes,
                     "ms_per_launch": ms_evolve, "share_of_step": ms_evolve * args.steps / ms_total,
                     # the whole step against the same peak: 88 B per particle + 72 B per event (the parent's
                     # momentum and optical depth rewritten = 32, the photon = 32, its parent index = 8; the records the two
                     # passes exchange are the implementation's traffic, not the method's)
                     "whole_step": {"algorithmic_bytes": step_bytes,
                                    "achieved": step_bytes / (ms_total / args.steps * 1e-3) / 1e9,
                                    "frac": step_bytes / (ms_total / args.steps * 1e-3) / 1e9 / peaks["hbm_gbs"]}},
        "kernels_ms": {"qed_step": {"evolve_pass": ms_evolve, "event_pass": ms_events},
                       "two_call_path": {"evolve_optical_depth": ms_evolve2, "generate_photons": ms_events2},
                       "two_call_path_stage_records": {"evolve_optical_depth": ms_evolve3, "generate_photons": ms_events3}},
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "steps": args.e2e_steps},
        "gpu_launches": 3 * args.steps,
        "clocks": sampler.summary(),
    }
    if not args.no_cpu_baseline and world == 1:
        tables = [ctx.export_tables(k) for k in range(4)]
        ns = min(args.cpu_sample, n)
        steps_cpu = 6  # 8 Mi x 6 particle-steps: 10-15 s on 16 host cores
        v, sec, threads = time_oracle(tp_kwargs, tables, ns, steps_cpu, dt)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle",
                                "sample": "first %d particles of the workload x %d steps (evolve + photon emission), "
                                          "%.1f s" % (ns, steps_cpu, sec)}
    if world == 1 and not args.no_other_configs:
        # the fp32 half of the metric (configs 3 and 5) and the table build (config 4), measured in the same run
        del p, fields, tau, ph_p, ph_tau, ph_parent, p_pin, field_pin, tau_pin, p_e2e, sec_pin
        torch.cuda.empty_cache()
        others = []
        for fn in (run_config3, run_config5):
            ctx_o = q.Context(local)
            for kv in args.opt:
                name, value = kv.split("=")
                ctx_o.set_option(name, int(value))
            ctx_o.build_tables(q.TableParams(**w.table_params(3)))
            others.append(fn(args, torch, q, w, ctx_o, dev, peaks, peak_kind))
            ctx_o.close()
            torch.cuda.empty_cache()
        others.append(run_config4(args, torch, q, w, peaks))
        line["other_configs"] = others
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_cascade(args):
    """closed loop in a uniform field (Ridgers case (iii): gamma_0 = 1000, B_0 = 9e-3 E_s/c, 0.1 fs in
    `steps` steps, photons below 2 m_e c^2 dropped at creation): push + QED step of the three species + feedback per
    step, populations growing from `particles`/2 electrons to ~4.4x as many particles.  Not the headline metric."""
    import torch

    import paper_2110_00256_b200 as q
    torch.cuda.set_device(0)
    ctx = q.Context(0)
    ctx.build_tables(q.TableParams())          # the paper's benchmark tables, 256 / 256x256
    dt_ = torch.float64 if args.cascade_dtype == "f64" else torch.float32
    n0 = args.particles // 2
    steps = max(args.steps, 1)

    def run():
        pops = {k: q.Species(6 * n0, dt_, dt_, ib)
                for k, ib in (("electrons", 0), ("positrons", 1 << 40), ("photons", 1 << 41))}
        pops["electrons"].p[0][:n0] = float(np.sqrt(1000.0 ** 2 - 1))
        pops["electrons"].n = n0
        ctx.init_optical_depth(q.LEPTON, pops["electrons"].tau[:n0], SEED, 0)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        work = 0
        for s in range(steps):
            work += sum(p.n for p in pops.values())
            ctx.cascade_step(pops, (0.0, 0.0, 0.0), (0.0, 0.0, 9e-3), 1e-16 / steps, SEED, s, photon_min_energy=2.0)
        torch.cuda.synchronize()
        return work, time.perf_counter() - t0, {k: p.n for k, p in pops.items()}

    for _ in range(max(1, min(args.warmup, 2))):
        run()                                  # scratch buffers reach their final size
    work, sec, final = run()
    print(json.dumps({"metric": "closed loop (Ridgers case iii) particle-steps/s", "value": work / sec,
                      "unit": "particle-steps/s", "n_gpus": 1, "steps": steps, "warmup": args.warmup,
                      "ms_per_step": 1e3 * sec / steps, "higher_is_better": True, "dtype": args.cascade_dtype,
                      "data": "synthetic",
                      "config": {"workload": "closed loop, uniform B = 9e-3 E_s/c, gamma_0 = 1000, 0.1 fs, photon "
                                             "threshold 2 m_e c^2", "initial_electrons": n0, "final": final}}), flush=True)


def run_tables(args):
    """BASELINE config 4 alone (the entry `other_configs` carries in the default run), as its own JSON line"""
    import torch

    import paper_2110_00256_b200 as q
    from paper_2110_00256_b200 import workloads as w
    torch.cuda.set_device(0)
    peaks, _ = measured_peaks()
    leg = run_config4(args, torch, q, w, peaks)
    line = {"metric": "table build time (BASELINE config 4)", "value": leg["value"], "unit": "ms", "n_gpus": 1, "steps": 5,
            "warmup": 2, "ms_per_step": leg["value"], "higher_is_better": False, "dtype": "f64", "data": "synthetic",
            "config": {"workload": leg["workload"], "cells": leg["cells"], "cells_per_s": leg["cells_per_s"],
                       "quadrature_kernels_ms": leg["quadrature_kernels_ms"]}}
    for k in ("roofline", "cpu_baseline"):
        if k in leg:
            line[k] = leg[k]
    print(json.dumps(line), flush=True)


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    elif args.tables:
        run_tables(args)
    elif args.cascade:
        run_cascade(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
