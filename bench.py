#!/usr/bin/env python
"""bench.py -- histories/s of the VPMC hot path on B200 (BASELINE.json metric) + seconds per dose at 0.5 %.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

A "step" is one pass of the whole hot path (S1-S6b + dose conversion + batch-uncertainty passes) over one batch of
synthetic input: the 8 plans of BASELINE.json configs[1] (water 100x100x150 @ 2 mm, 30 mm brass with a 1/2/3/4 cm
opening, each with and without a 45 mm WET range shifter, 825-3993 spots, 10^7 histories per plan = 8x10^7 per step).
`value` = histories/s with every input resident in HBM; `e2e` = the same through the C-ABI with host buffers
(vpmc_create + set_* from pinned host arrays, vpmc_dose_host back to pinned host memory, vpmc_destroy).
N > 1 (torchrun): every rank runs the same plans under its own Philox key (weak scaling) and the dose grids are
averaged with one NCCL all-reduce per plan.  `--impl reference` times the CPU oracle instead.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "proton histories/s"
SEED = 2
# The path is bound by plain ALU / MUFU instruction issue.  Unit of work = one material step of one history;
# per-unit figure = USEFUL lane-instructions of that step (step physics + Philox + rotation + move + the stage's geometry),
# from the committed ncu source-level counts (profiles/r1_*): overhead passes (refill, bookkeeping, idle lanes) are
# deliberately not counted, so `frac` is the fraction of the issue peak spent on the method's arithmetic.
INST_PER_SLAB_STEP = 450.0            # beam_kernel: range-shifter / brass step
INST_PER_CT_STEP = 510.0              # voxel_kernel: voxel step incl. face distance, material fetch, scoring
ALG_BYTES_PER_CT_STEP = 10.0          # 2 B HU read + 4 B read + 4 B write of the dose add
ALG_BYTES_PER_HISTORY_BEAM = 48.0     # source record read; + 80 B queue record written per survivor
# DRAM traffic per history of the two kernels, from the ncu --set full capture (profiles/r1_ncu_full.md)
DRAM_BYTES_PER_HISTORY = {"beam_kernel": 63.0, "voxel_kernel": 22.0}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", 1965.0)), "measured"
    return 6650.0, 1965.0, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.idx = gpu_index
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is not None:
            self.p.terminate()
            try:
                self.p.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 8 or not c[0].isdigit() or int(c[0]) != self.idx:
                continue
            try:
                sm.append(float(c[1])); mx.append(float(c[2]))
            except ValueError:
                continue
            for n, v in zip(names, c[4:8]):
                if v == "Active":
                    reasons.add(n)
        self.f.close()
        os.unlink(self.f.name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "reasons": sorted(reasons), "samples": len(sm)}


def pinned(a):
    """numpy view of a pinned host copy of array a."""
    import torch
    t = torch.from_numpy(a.copy()).pin_memory()
    return t.numpy()


def pin_problem(w):
    w = dict(w)
    w["ct"] = dict(w["ct"]); w["ct"]["hu"] = pinned(w["ct"]["hu"])
    beams = []
    for b in w["beams"]:
        b = dict(b); b["spots"] = pinned(b["spots"])
        if b.get("aperture") is not None:
            b["aperture"] = dict(b["aperture"]); b["aperture"]["open"] = pinned(b["aperture"]["open"])
        beams.append(b)
    w["beams"] = beams
    return w


def workload_plans(args):
    """(label, workloads function name, kwargs) of the plans one step runs, and the default histories per plan."""
    from paper_2307_01416_b200 import workloads as wl
    if args.workload == "config2":
        plans = wl.config2_plans()
        if args.plans:
            plans = [(int(x.split(":")[0]), bool(int(x.split(":")[1]))) for x in args.plans.split(",")]
        return [("d%d_%s" % (d, "rs" if rs else "nors"), "config2", {"opening_mm": d, "range_shifter": rs}) for (d, rs) in plans], 10_000_000, \
            "BASELINE.json configs[1]: water 100x100x150 @ 2 mm, 8 plans (opening 1/2/3/4 cm x RS off/on), 825-3993 spots"
    if args.workload == "config3":
        return [("seed%d" % s, "config3", {"seed": s}) for s in (3, 4, 5, 6)], 10_000_000, \
            "BASELINE.json configs[2]: synthetic head CT 256x256x160 @ 1x1x1.5 mm, 2 beams, apertures = target + 3 mm, 4 patients (seeds 3-6)"
    if args.workload == "config5":
        return [("stress", "config5", {})], 100_000_000, \
            "BASELINE.json configs[4]: 512x512x200 @ 1 mm random-slab phantom, RS 45 mm + star-shaped aperture, 70-230 MeV"
    raise SystemExit("unknown --workload %s" % args.workload)


def run_reference(args):
    """The CPU oracle on the same workload/metric; each step = a bounded sample of the plans."""
    from oracle import cpu_bench
    from paper_2307_01416_b200 import workloads as wl
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    plans, n_default, label = workload_plans(args)
    if args.histories <= 0:
        args.histories = n_default
    per_plan = args.ref_sample // len(plans)
    rates, cores = [], cpu_bench.n_cores()
    t_all = []
    for it in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        done, busy = 0, 0.0
        for (_, fn, kw) in plans:
            r, cores, _ = cpu_bench.time_oracle(fn, kw, args.histories, SEED, per_plan)
            busy += per_plan / r
            done += per_plan
        if it >= args.warmup:
            rates.append(done / busy)
            t_all.append(time.perf_counter() - t0)
    v = sum(rates) / len(rates)
    sample = "%d histories per plan over %d plans per step, ids spread over the %d-history run" % (per_plan, len(plans), args.histories)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": "histories/s", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * sum(t_all) / len(t_all), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": label + " (bounded sample)", "histories_per_plan": args.histories},
        "cpu_baseline": {"value": v, "unit": "histories/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": "histories/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200")
    ap.add_argument("--workload", default="config2", help="config2 (default, the bench workload) | config3 | config5 | config4 (influence build)")
    ap.add_argument("--histories", type=int, default=0, help="histories per plan (0 = the config's own: 1e7, 1e8 for config5)")
    ap.add_argument("--hist-per-spot", type=int, default=10_000, help="config4: histories per spot and scenario")
    ap.add_argument("--ref-sample", type=int, default=800_000, help="oracle histories per reference step")
    ap.add_argument("--cpu-sample", type=int, default=1_600_000, help="oracle histories of the cpu_baseline leg")
    ap.add_argument("--plans", default="", help="subset of the 8 plans as opening_mm:rs pairs, e.g. 20:0,20:1 (profiling)")
    ap.add_argument("--n-batches", type=int, default=10, help="batches of the uncertainty estimate (vpmc_params.n_batches)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-dose-at-unc", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.workload == "config4":
        return run_influence(args)
    run_b200(args)


# run_b200 is appended below


def run_b200(args):
    import numpy as np
    import torch
    from paper_2307_01416_b200 import binding, dist, workloads as wl

    rank, local_rank, world = dist.init()
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    hbm_gbs, sm_max_mhz, peak_kind = load_peaks()
    plans, n_default, label = workload_plans(args)
    N = int(args.histories) if args.histories > 0 else n_default
    seed = dist.rank_seed(SEED, rank)
    problems = [getattr(wl, fn)(**kw) for (_, fn, kw) in plans]
    params = binding.default_params(n_batches=args.n_batches)

    # ---- set-up (S0), not part of histories/s
    t0 = time.perf_counter()
    engines = [binding.Engine(p, params) for p in problems]
    doses = [torch.empty(e.nvox, dtype=torch.float32, device=dev) for e in engines]
    torch.cuda.synchronize()
    setup_s = time.perf_counter() - t0
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)     # > 126 MB L2
    stream = torch.cuda.current_stream()

    def step():
        for e, d in zip(engines, doses):
            e.dose(N, seed, out=d, stream=stream)
            dist.combine_dose(d, world)

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    for e in engines:
        e.set_timing(True)
        e.timing()
    launches0 = sum(e.launch_count() for e in engines)
    dist.barrier(world)
    torch.cuda.synchronize()
    sampler = ClockSampler(torch.cuda.current_device() if "CUDA_VISIBLE_DEVICES" not in os.environ else local_rank)
    sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for k in range(args.steps):
        flush.zero_()                                   # L2 flush between timed iterations (not timed)
        ev[k][0].record(stream)
        step()
        ev[k][1].record(stream)
    torch.cuda.synchronize()
    dist.barrier(world)
    clocks = sampler.stop()
    t_ms = sum(a.elapsed_time(b) for a, b in ev)
    t_ms = dist.max_over_ranks(t_ms, world, dev)
    launches = sum(e.launch_count() for e in engines) - launches0
    hist_per_step = N * len(plans) * world
    value = hist_per_step * args.steps / (t_ms * 1e-3)

    # ---- roofline of the dominant kernel, live CUDA-event durations from the library (events on the launching stream)
    tm = {"beamline": [0.0, 0], "voxel": [0.0, 0], "scoring": [0.0, 0], "writer": [0.0, 0]}
    steps_ct = steps_slab = n_surv = 0
    for e in engines:
        for k, (ms, n) in e.timing().items():
            tm[k][0] += ms; tm[k][1] += n
        e.set_timing(False)
        tl = e.tallies()                                 # of the last dose() call = one timed step's share
        steps_ct += tl.n_steps_ct; steps_slab += tl.n_steps_slab
        n_surv += tl.n_stopped_ct + tl.n_nuclear + tl.n_escaped     # upper bound of the histories that reached the CT
    peak_ginst = 148 * 4 * 32 * sm_max_mhz * 1e6 / 1e9        # lane-instructions/s at the max SM clock

    def kernel_roofline(name, cls, inst_per_unit, units_per_step, alg_bytes_per_step):
        ms, n = tm[cls]
        launches = max(n, 1)
        avg_s = ms * 1e-3 / launches
        units = units_per_step * args.steps / launches
        ach = inst_per_unit * units / avg_s / 1e9 if avg_s > 0 else 0.0
        hist_per_launch = N * len(plans) * args.steps / launches
        return {"kernel": name, "bound": "alu", "achieved": ach, "peak": peak_ginst, "unit": "Glane-inst/s", "frac": ach / peak_ginst,
                "traffic": DRAM_BYTES_PER_HISTORY[name] * hist_per_launch, "inst_per_unit": inst_per_unit, "units_per_launch": units,
                "avg_launch_ms": avg_s * 1e3, "launches": n, "share_of_step": ms / max(t_ms, 1e-9),
                "hbm": {"achieved": alg_bytes_per_step * args.steps / launches / avg_s / 1e9 if avg_s > 0 else 0.0, "peak": hbm_gbs, "unit": "GB/s",
                        "frac": (alg_bytes_per_step * args.steps / launches / avg_s / 1e9 / hbm_gbs) if avg_s > 0 else 0.0,
                        "peak_source": peak_kind + " MEASURED_PEAKS.json hbm_gbs"}}

    kr = [kernel_roofline("beam_kernel", "beamline", INST_PER_SLAB_STEP, steps_slab, ALG_BYTES_PER_HISTORY_BEAM * N * len(plans) + 80.0 * n_surv),
          kernel_roofline("voxel_kernel", "voxel", INST_PER_CT_STEP, steps_ct, ALG_BYTES_PER_CT_STEP * steps_ct + 80.0 * n_surv)]
    dom = max(kr, key=lambda r: r["share_of_step"])
    roofline = dict(dom)
    roofline["peak_source"] = "148 SM x 4 SMSP x 32 lanes x %.0f MHz (%s sm_max_mhz); DESIGN.md 7" % (sm_max_mhz, peak_kind)
    roofline["note"] = ("timed classes: beamline = source_kernel + beam_kernel, voxel = entry_kernel + voxel_kernel; the one-thread-per-item "
                        "source / entry kernels are < 5 % of their class (profiles/r1_launches.md)")
    roofline["other_kernels"] = [r for r in kr if r is not dom]
    roofline["share_of_step"] = {k: v[0] / max(t_ms, 1e-9) for k, v in tm.items()}

    # ---- e2e: host buffers in, host dose out, through the C-ABI, H2D/D2H inside the timed region
    pinned_problems = [pin_problem(p) for p in problems]
    host_out = [pinned(np.empty(e.nvox, dtype=np.float32)) for e in engines]
    for e in engines:
        e.close()
    del engines

    def e2e_step():
        h2d = d2h = 0
        for p, out in zip(pinned_problems, host_out):
            e = binding.Engine(p, params)
            e.dose_host(N, seed, out=out)
            h2d += e.h2d_bytes; d2h += out.nbytes
            e.close()
        return h2d, d2h

    for _ in range(2):                                   # warm-up: allocator cache, page-locked staging
        e2e_step()
    dist.barrier(world)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        h2d, d2h = e2e_step()
    torch.cuda.synchronize()
    e2e_s = dist.max_over_ranks(time.perf_counter() - t0, world, dev)
    e2e = {"value": hist_per_step * args.steps / e2e_s, "unit": "histories/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h}

    out = {"metric": METRIC, "value": value, "unit": "histories/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": t_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f32", "data": "synthetic",
           "config": {"workload": label, "histories_per_plan": N, "plans_per_step": len(plans),
                      "n_batches": args.n_batches, "l2_flush_between_steps": True, "parallelism": "replicas x%d + dose all-reduce" % world,
                      "setup_s": setup_s},
           "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline}

    if rank == 0 and world == 1 and not args.no_dose_at_unc and args.workload == "config2":
        out["dose_at_0p5pct"] = dose_at_uncertainty(binding, wl)
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import cpu_bench
        per_plan = args.cpu_sample // len(plans)
        busy, done, cores = 0.0, 0, 1
        for (_, fn, kw) in plans:
            r, cores, _ = cpu_bench.time_oracle(fn, kw, N, SEED, per_plan)
            busy += per_plan / r; done += per_plan
        out["cpu_baseline"] = {"value": done / busy, "unit": "histories/s", "cores": cores, "kind": "oracle",
                               "sample": "%d histories per plan over the %d plans, ids spread over the %d-history run, "
                                         "%d single-threaded oracle processes" % (per_plan, len(plans), N, cores)}
    if rank == 0:
        print(json.dumps(out))


def dose_at_uncertainty(binding, wl, target=0.005):
    """Second half of the metric: seconds per dose at 0.5 % statistical uncertainty (SURVEY.md 8(c)-C6 estimator):
    set-up + a pilot run + the run sized from the pilot by N = N0 (u0/target)^2; the final run's own estimate is reported."""
    import torch
    p = wl.config2(20, False)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    e = binding.Engine(p)
    n0 = 1_000_000
    d = e.dose(n0, SEED)
    u0 = e.uncertainty()
    n = int(min(max(n0 * (u0 / target) ** 2 * 1.05, n0), 2e9))
    d = e.dose(n, SEED + 1, out=d)
    u = e.uncertainty()
    torch.cuda.synchronize()
    sec = time.perf_counter() - t0
    e.close()
    return {"workload": "config2 opening 2 cm, no range shifter", "seconds": sec, "histories": n + n0, "uncertainty": u,
            "pilot_uncertainty": u0, "target": target}




def run_influence(args):
    """--workload config4: the 13-scenario influence-matrix build (S7 + S8) on the config-3 head with ~2000 spots."""
    import torch
    from paper_2307_01416_b200 import binding, workloads as wl
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(0)
    w = wl.config4(hist_per_spot=args.hist_per_spot)
    eng = binding.Engine(w)
    sc = [binding.scenario(s, k) for s, k in w["scenarios"]]
    hps = int(args.hist_per_spot)

    def step():
        res = eng.influence(sc, hps, w["rel_threshold"], SEED)
        nnz = sum(int(c.numel()) for (_, c, _) in res)
        del res
        return nnz

    for _ in range(max(args.warmup, 1)):
        step()
    torch.cuda.synchronize()
    eng.set_timing(True); eng.timing()
    l0 = eng.launch_count()
    sampler = ClockSampler(torch.cuda.current_device()); sampler.start()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(args.steps):
        nnz = step()
    b.record(); torch.cuda.synchronize()
    clocks = sampler.stop()
    t_ms = a.elapsed_time(b)
    tm = eng.timing()
    n_hist = len(sc) * eng.n_spots * hps
    out = {"metric": METRIC, "value": n_hist * args.steps / (t_ms * 1e-3), "unit": "histories/s", "n_gpus": 1, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": t_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f32", "data": "synthetic",
           "config": {"workload": "BASELINE.json configs[3]: 13-scenario influence matrices on the config-3 head (%s), %d spots, "
                                  "%d histories per spot, threshold 1e-4" % (w["name"], eng.n_spots, hps),
                      "seconds_per_13_matrices": t_ms * 1e-3 / args.steps, "nnz_total": nnz, "csr_bytes": nnz * 8 + 13 * (eng.n_spots + 1) * 8,
                      "l2_flush_between_steps": False, "inputs_larger_than_l2": True},
           "clocks": clocks, "gpu_launches": eng.launch_count() - l0,
           "share_of_step": {k: v[0] / t_ms for k, v in tm.items()}}
    eng.close()
    print(json.dumps(out))


if __name__ == "__main__":
    main()
