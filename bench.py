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
# dram__bytes_read.sum + dram__bytes_write.sum of one launch of the evolve pass (16 Mi particles), ncu --set full:
# profiles/r1d_step_full.md (1.343606 GB read = the 80 B/particle of inputs; 109 MB written: part of the 134 MB of
# new tau is still dirty in L2 when the kernel ends, plus the staged records)
EVOLVE_DRAM_TRAFFIC_BYTES = 1343606000 + 108954112


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
    # bound the run: at ~4e6 particle-steps/s an 8 Mi sample takes ~2 s per step
    steps_run = min(steps, 8)
    value, sec, threads = time_oracle(tp, tables, n, steps_run, dt)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": steps_run,
            "warmup": args.warmup, "ms_per_step": 1e3 * sec / steps_run, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "config 2 (synchrotron emission, fp64), oracle on host cores", "particles": n,
                       "tables": "1024 / 1024x1024 (stand-in values, same shape)"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle",
                             "sample": "%d particles x %d steps (evolve + photon emission)" % (n, steps_run)},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


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
                     "traffic": EVOLVE_DRAM_TRAFFIC_BYTES, "algorithmic_bytes_per_launch": evolve_bytes,
                     "ms_per_launch": ms_evolve, "share_of_step": ms_evolve * args.steps / ms_total,
                     # the whole step against the same peak: 88 B per particle + 168 B per event (48 B record written and
                     # read back once = 96, 32 B photon + 8 B parent index, four 8-byte parent stores = 32: DESIGN.md 6)
                     "whole_step": {"algorithmic_bytes": evolve_bytes + 168 * fired_last,
                                    "achieved": (evolve_bytes + 168 * fired_last) / (ms_total / args.steps * 1e-3) / 1e9,
                                    "frac": (evolve_bytes + 168 * fired_last) / (ms_total / args.steps * 1e-3) / 1e9
                                            / peaks["hbm_gbs"]}},
        "kernels_ms": {"qed_step": {"evolve_pass": ms_evolve, "event_pass": ms_events},
                       "two_call_path": {"evolve_optical_depth": ms_evolve2, "generate_photons": ms_events2}},
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
    """BASELINE config 4: picsarqed_build_tables on 4096 log-spaced chi points over [1e-4, 1e3], 2048 xi columns,
    both processes (the 2D tables carry all 4096 rows: DESIGN.md 4).  Time per build, median of `steps`."""
    import torch

    import paper_2110_00256_b200 as q
    from paper_2110_00256_b200 import workloads as w
    torch.cuda.set_device(0)
    ctx = q.Context(0)
    tp = q.TableParams(**w.table_params(4))
    times = []
    for _ in range(max(1, args.warmup) + max(1, min(args.steps, 10))):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        ctx.build_tables(tp)                      # synchronises
        times.append(time.perf_counter() - t0)
    ms = 1e3 * float(np.median(times[max(1, args.warmup):]))
    cells = 2 * tp.qs_n_chi * tp.qs_n_xi
    print(json.dumps({"metric": "table build time (BASELINE config 4)", "value": ms, "unit": "ms", "n_gpus": 1,
                      "steps": len(times) - max(1, args.warmup), "warmup": max(1, args.warmup), "ms_per_step": ms,
                      "higher_is_better": False, "dtype": "f64", "data": "synthetic",
                      "config": {"workload": "4096-point lnG, lnT on [1e-4, 1e3]; two 4096 x 2048 CDF tables",
                                 "cells": cells, "cells_per_s": cells / (ms * 1e-3)}}), flush=True)


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
