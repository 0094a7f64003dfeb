#!/usr/bin/env python
"""bench.py -- histories/s of the VPMC hot path on B200 (BASELINE.json metric) + seconds per dose at 0.5 %.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload config5|config2|config3|config4]

A "step" is one pass of the whole hot path (S1-S6b + dose conversion + batch-uncertainty passes) over one batch of
synthetic input.  The default workload is the largest single-GPU configuration of BASELINE.json: configs[4], the 512x512x200
@ 1 mm random-slab phantom behind a 45 mm range shifter and a star-shaped brass aperture, 10^8 histories per step.
`value` = histories/s with every input resident in HBM; `e2e` = the same through the C-ABI with host buffers (vpmc_create +
set_* from pinned host arrays, vpmc_dose_host back to pinned host memory, vpmc_destroy).  At N = 1 the same run also measures
the other configurations as sub-records under `configs`: configs[1] (8 water plans x 10^7), configs[2] (head CT, >= 10 seeds,
each run to 0.5 % with the stopping rule on the device) and configs[3] (13 influence matrices).
N > 1 (torchrun): rank r transports shard r of N of every spot's history ids of the SAME (N x 10^8)-history run and the dose
grids are summed with one all-reduce; weak scaling.  `--impl reference` times the CPU oracle instead.
"""
from __future__ import annotations

import argparse
import csv
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
# The path is bound by plain ALU / MUFU instruction issue.  Unit of work = one material step of one history.
# Thread-instructions per unit are MEASURED: ncu's smsp__thread_inst_executed.sum over every launch of a kernel divided by
# the steps the kernels counted in the same run (profiles/r2_inst_per_step.csv, written by `bench.py --ncu-summary`, one row
# per config and kernel; it counts everything the kernel executes -- refill, bookkeeping, idle lanes included).  The survey's
# own estimate of the method's arithmetic (350-400 per step) is reported beside it.
INST_CSV = os.path.join(ROOT, "profiles", "r2_inst_per_step.csv")
SURVEY_INST_PER_STEP = 375.0
ALG_BYTES_PER_CT_STEP = 10.0          # 2 B HU read + 4 B read + 4 B write of the dose add


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
            b["aperture"] = dict(b["aperture"])
            for k in ("open", "polygon"):
                if b["aperture"].get(k) is not None:
                    b["aperture"][k] = pinned(b["aperture"][k])
        beams.append(b)
    w["beams"] = beams
    return w


CONFIG3_SEEDS = (3, 4, 5, 6, 7, 8, 9, 10, 11, 12)


def workload_plans(name, plans_arg=""):
    """(label, workloads function name, kwargs) of the plans one step runs, the default histories per plan, a description."""
    from paper_2307_01416_b200 import workloads as wl
    if name == "config2":
        plans = wl.config2_plans()
        if plans_arg:
            plans = [(int(x.split(":")[0]), bool(int(x.split(":")[1]))) for x in plans_arg.split(",")]
        return [("d%d_%s" % (d, "rs" if rs else "nors"), "config2", {"opening_mm": d, "range_shifter": rs}) for (d, rs) in plans], 10_000_000, \
            "BASELINE.json configs[1]: water 100x100x150 @ 2 mm, 8 plans (opening 1/2/3/4 cm x RS off/on), 825-3993 spots"
    if name == "config3":
        return [("seed%d" % s, "config3", {"seed": s}) for s in CONFIG3_SEEDS[:4]], 10_000_000, \
            "BASELINE.json configs[2]: synthetic head CT 256x256x160 @ 1x1x1.5 mm, 2 beams, apertures = target + 3 mm, 4 patients (seeds 3-6)"
    if name == "config5":
        return [("stress", "config5", {})], 100_000_000, \
            "BASELINE.json configs[4]: 512x512x200 @ 1 mm random-slab phantom, RS 45 mm + star-shaped aperture, 70-230 MeV"
    if name == "config5_polygon":
        return [("stress_polygon", "config5", {"polygon": True})], 100_000_000, \
            "BASELINE.json configs[4] with the star-shaped opening given as its 720-vertex boundary polygon (crossing-number test on the device, SURVEY.md 8(f)-2)"
    raise SystemExit("unknown --workload %s" % name)


def run_reference(args):
    """The CPU oracle on the same workload/metric; each step = a bounded sample of the plans."""
    from oracle import cpu_bench
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    plans, n_default, label = workload_plans(args.workload if args.workload != "config4" else "config3", args.plans)
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
    ap.add_argument("--workload", default="config5", help="config5 (default: the largest single-GPU config) | config2 | config3 | config4 (influence build)")
    ap.add_argument("--histories", type=int, default=0, help="histories per plan (0 = the config's own: 1e8 for config5, else 1e7)")
    ap.add_argument("--hist-per-spot", type=int, default=10_000, help="config4: histories per spot and scenario")
    ap.add_argument("--ref-sample", type=int, default=800_000, help="oracle histories per reference step")
    ap.add_argument("--cpu-sample", type=int, default=1_600_000, help="oracle histories of the cpu_baseline leg")
    ap.add_argument("--plans", default="", help="config2: subset of the 8 plans as opening_mm:rs pairs, e.g. 20:0,20:1 (profiling)")
    ap.add_argument("--n-batches", type=int, default=10, help="batches of the uncertainty estimate (vpmc_params.n_batches)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-subrecords", action="store_true", help="skip the configs[1..3] sub-records (profiling runs)")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (profiling runs only: the line then has no e2e)")
    ap.add_argument("--ncu-summary", nargs=3, metavar=("NCU_CSV", "BENCH_LOG", "CONFIG"),
                    help="no GPU work: turn an ncu --csv metrics log of a bench run + that run's stdout into rows of " + os.path.relpath(INST_CSV, ROOT))
    args = ap.parse_args()
    if args.ncu_summary:
        return ncu_summary(*args.ncu_summary)
    if args.impl == "reference":
        return run_reference(args)
    if args.workload == "config4":
        import torch
        assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
        torch.cuda.set_device(0)
        out = measure_influence(args.hist_per_spot, args.steps, max(args.warmup, 1))
        out.update({"metric": METRIC, "unit": "histories/s", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
                    "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic"})
        print(json.dumps(out))
        return
    run_b200(args)


# ------------------------------------------------------------------------------------------- measured instruction counts
def load_inst_counts(config):
    """{kernel: row} of profiles/r2_inst_per_step.csv for one config (None if the file has no such rows)."""
    if not os.path.exists(INST_CSV):
        return None
    rows = {r["kernel"]: r for r in csv.DictReader(open(INST_CSV)) if r["config"] == config}
    return rows or None


def ncu_summary(ncu_csv, bench_log, config):
    """Per kernel of one profiled bench run: thread / warp instructions, DRAM and L2 bytes, RED sectors, all divided by the
    material steps the kernels counted in that run (the bench line printed by the same process)."""
    import collections
    import re
    line = [l for l in open(bench_log) if l.startswith("{")][-1]
    b = json.loads(line)
    if config == "config4":
        # influence build: only the MODE 1 voxel kernel (private boxes) counts its steps in the tallies; the pilot (MODE 2) does not
        calls = b["profile_units"]["builds_run"]
        units = {"voxel_kernel_box": b["profile_units"]["ct_steps_per_build"] * calls}
    else:
        calls = b["profile_units"]["steps_run"]          # the profiled run must be --no-e2e --no-subrecords: nothing else launches these kernels
        units = {"beam_kernel": b["profile_units"]["slab_steps_per_step"] * calls, "voxel_kernel": b["profile_units"]["ct_steps_per_step"] * calls}
    acc = collections.defaultdict(lambda: collections.defaultdict(float))
    for r in csv.DictReader(l for l in open(ncu_csv) if l.startswith('"')):
        name = re.sub(r"^void ", "", r["Kernel Name"])
        name = re.sub(r"^vpk::", "", name)
        if config == "config4" and re.match(r"voxel_kernel<(\(int\))?1,", name):
            name = "voxel_kernel_box"
        name = re.sub(r"[<(].*", "", name)
        try:
            v = float(r["Metric Value"].replace(",", ""))
        except ValueError:
            continue
        acc[name][r["Metric Name"]] += v
        if r["Metric Name"] == "gpu__time_duration.sum":
            acc[name]["launches"] += 1
    fields = ["config", "kernel", "launches", "time_ms", "units", "thread_inst_per_unit", "warp_inst_per_unit", "lanes_per_inst",
              "dram_bytes_per_unit", "l2_bytes_per_unit", "red_sectors_per_unit", "l2_hit_pct"]
    old = []
    if os.path.exists(INST_CSV):
        old = [r for r in csv.DictReader(open(INST_CSV)) if r["config"] != config]
    rows = []
    for k, u in units.items():
        d = acc.get(k)
        if not d or not u:
            continue
        rows.append({"config": config, "kernel": k, "launches": int(d["launches"]), "time_ms": "%.3f" % (d["gpu__time_duration.sum"] / 1e6),
                     "units": int(u), "thread_inst_per_unit": "%.2f" % (d["smsp__thread_inst_executed.sum"] / u),
                     "warp_inst_per_unit": "%.3f" % (d["smsp__inst_executed.sum"] / u),
                     "lanes_per_inst": "%.2f" % (d["smsp__thread_inst_executed.sum"] / max(d["smsp__inst_executed.sum"], 1.0)),
                     "dram_bytes_per_unit": "%.3f" % ((d["dram__bytes_read.sum"] + d["dram__bytes_write.sum"]) / u),
                     "l2_bytes_per_unit": "%.2f" % (d["lts__t_bytes.sum"] / u),
                     "red_sectors_per_unit": "%.3f" % (d["lts__t_sectors_op_red.sum"] / u),
                     "l2_hit_pct": "%.1f" % (d["lts__t_sector_hit_rate.pct"] / max(d["launches"], 1.0))})
    with open(INST_CSV, "w", newline="") as f:
        wr = csv.DictWriter(f, fieldnames=fields)
        wr.writeheader()
        for r in old + rows:
            wr.writerow(r)
    print("wrote %d rows for %s to %s" % (len(rows), config, INST_CSV))


# ------------------------------------------------------------------------------------------- dose workloads
def measure_dose(workload, args, rank, local_rank, world, dev, steps, warmup, with_e2e, e2e_warmup=1):
    """Times `steps` steps of a dose workload (all its plans, N histories each) resident in HBM, then (with_e2e) the same
    through host buffers.  Returns the record (value, ms_per_step, per-class timing, step counts, e2e)."""
    import numpy as np
    import torch
    from paper_2307_01416_b200 import binding, dist, workloads as wl
    plans, n_default, label = workload_plans(workload, args.plans)
    N = int(args.histories) if (args.histories > 0 and workload == args.workload) else n_default
    problems = [getattr(wl, fn)(**kw) for (_, fn, kw) in plans]
    params = binding.default_params(n_batches=args.n_batches)

    t0 = time.perf_counter()                              # set-up (S0), not part of histories/s
    engines = [binding.Engine(p, params) for p in problems]
    doses = [torch.empty(e.nvox, dtype=torch.float32, device=dev) for e in engines]
    torch.cuda.synchronize()
    setup_s = time.perf_counter() - t0
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)     # > 126 MB L2
    stream = torch.cuda.current_stream()

    def step():
        for e, d in zip(engines, doses):
            dist.sharded_dose(e, N * world, SEED, rank, world, out=d, stream=stream)

    for _ in range(warmup):
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
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for k in range(steps):
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
    tm = {k: [0.0, 0] for k in ("beamline", "voxel", "scoring", "writer", "stage", "optimiser")}
    steps_ct = steps_slab = 0
    finite = True
    for e, d in zip(engines, doses):
        for k, (ms, n) in e.timing().items():
            tm[k][0] += ms; tm[k][1] += n
        e.set_timing(False)
        tl = e.tallies()                                 # of the last dose() call = one timed step's share of this rank
        steps_ct += tl.n_steps_ct; steps_slab += tl.n_steps_slab
        finite = finite and bool(torch.isfinite(d).all())
    rec = {"workload": label, "value": hist_per_step * steps / (t_ms * 1e-3), "ms_per_step": t_ms / steps, "histories_per_plan": N * world,
           "plans_per_step": len(plans), "setup_s": setup_s, "gpu_launches": launches, "clocks": clocks, "dose_finite": finite,
           "timing_ms_per_step": {k: v[0] / steps for k, v in tm.items()}, "launches_per_step": {k: v[1] / steps for k, v in tm.items()},
           "ct_steps_per_step": steps_ct, "slab_steps_per_step": steps_slab, "step_ms_total": t_ms, "steps": steps}
    assert finite, "non-finite dose"
    red = engines[0].bench_red(4 << 20, 1 << 29) if rank == 0 else None
    if with_e2e:
        pinned_problems = [pin_problem(p) for p in problems]
        host_out = [pinned(np.empty(e.nvox, dtype=np.float32)) for e in engines]
    for e in engines:
        e.close()
    del engines, doses, flush
    if with_e2e:
        # host buffers in, host dose out, through the C-ABI; H2D / D2H inside the timed region
        def e2e_step():
            h2d = d2h = 0
            for p, out in zip(pinned_problems, host_out):
                e = binding.Engine(p, params)
                e.set_shard(rank, world)
                e.dose_host(N * world, SEED, out=out)
                h2d += e.h2d_bytes; d2h += out.nbytes
                e.close()
            return h2d, d2h

        for _ in range(e2e_warmup):
            e2e_step()
        dist.barrier(world)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(steps):
            h2d, d2h = e2e_step()
        torch.cuda.synchronize()
        e2e_s = dist.max_over_ranks(time.perf_counter() - t0, world, dev)
        rec["e2e"] = {"value": hist_per_step * steps / e2e_s, "unit": "histories/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                      "warmup": e2e_warmup, "note": "per rank: this rank's shard; D2H of the rank's partial grid"}
    rec["red_ceiling"] = red
    return rec


def rooflines(rec, config, hbm_gbs, sm_max_mhz, peak_kind):
    """Per-kernel roofline records of a measure_dose() record: live CUDA-event durations x counted steps x measured instructions."""
    peak = 148 * 4 * 32 * sm_max_mhz * 1e6 / 1e9          # lane-instructions/s at the max SM clock, in G
    counts = load_inst_counts(config)
    out = []
    steps = rec["steps"]
    for name, cls, units in (("beam_kernel", "beamline", rec["slab_steps_per_step"]), ("voxel_kernel", "voxel", rec["ct_steps_per_step"])):
        ms = rec["timing_ms_per_step"][cls]
        n = rec["launches_per_step"][cls]
        if n <= 0 or ms <= 0:
            continue
        avg_s = ms * 1e-3 / n
        upl = units / n
        row = counts.get(name) if counts else None
        ipu = float(row["thread_inst_per_unit"]) if row else None
        ach = ipu * upl / avg_s / 1e9 if ipu else None
        surv = SURVEY_INST_PER_STEP * upl / avg_s / 1e9
        r = {"kernel": name, "bound": "alu", "achieved": ach, "peak": peak, "unit": "Glane-inst/s", "frac": (ach / peak) if ach else None,
             "frac_survey_count": surv / peak, "inst_per_unit": ipu, "inst_per_unit_survey": SURVEY_INST_PER_STEP,
             "inst_source": ("profiles/r2_inst_per_step.csv row (%s, %s): ncu smsp__thread_inst_executed.sum over all launches / steps counted "
                             "by the kernels; all instructions incl. refill and bookkeeping" % (config, name)) if row else "no committed ncu counts for this config",
             "lanes_per_inst": float(row["lanes_per_inst"]) if row else None,
             "units_per_launch": upl, "avg_launch_ms": avg_s * 1e3, "launches_per_step": n, "share_of_step": ms / rec["ms_per_step"],
             "traffic": float(row["dram_bytes_per_unit"]) * upl if row else None,
             "l2": {"bytes_per_unit": float(row["l2_bytes_per_unit"]), "achieved_GBps": float(row["l2_bytes_per_unit"]) * upl / avg_s / 1e9,
                    "hit_pct": float(row["l2_hit_pct"])} if row else None}
        if name == "voxel_kernel":
            alg = ALG_BYTES_PER_CT_STEP * upl
            r["hbm"] = {"achieved": alg / avg_s / 1e9, "peak": hbm_gbs, "unit": "GB/s", "frac": alg / avg_s / 1e9 / hbm_gbs,
                        "algorithmic_bytes_per_unit": ALG_BYTES_PER_CT_STEP, "peak_source": peak_kind + " MEASURED_PEAKS.json hbm_gbs"}
            if rec.get("red_ceiling"):
                ceil = rec["red_ceiling"][0]
                r["red"] = {"achieved_ops_per_s": upl / avg_s, "ceiling_ops_per_s": ceil, "frac": upl / avg_s / ceil,
                            "ceiling_source": "vpmc_bench_red: random fp32 atomicAdd into a 4 MB L2-resident buffer, measured in this run"}
        out.append(r)
    return out


def run_b200(args):
    import torch
    from paper_2307_01416_b200 import binding, dist

    rank, local_rank, world = dist.init()
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    hbm_gbs, sm_max_mhz, peak_kind = load_peaks()

    rec = measure_dose(args.workload, args, rank, local_rank, world, dev, args.steps, args.warmup, with_e2e=not args.no_e2e)
    kr = rooflines(rec, args.workload, hbm_gbs, sm_max_mhz, peak_kind)
    dom = max(kr, key=lambda r: r["share_of_step"])
    roofline = dict(dom)
    roofline["peak_source"] = "148 SM x 4 SMSP x 32 lanes x %.0f MHz (%s sm_max_mhz); DESIGN.md 7" % (sm_max_mhz, peak_kind)
    roofline["other_kernels"] = [r for r in kr if r is not dom]
    roofline["share_of_step"] = {k: v / rec["ms_per_step"] for k, v in rec["timing_ms_per_step"].items()}
    out = {"metric": METRIC, "value": rec["value"], "unit": "histories/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": rec["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f32", "data": "synthetic",
           "config": {"workload": rec["workload"], "histories_per_plan": rec["histories_per_plan"], "plans_per_step": rec["plans_per_step"],
                      "n_batches": args.n_batches, "l2_flush_between_steps": True,
                      "parallelism": "1 GPU" if world == 1 else "history-id shards x%d of one run + dose all-reduce (SUM)" % world,
                      "setup_s": rec["setup_s"]},
           "clocks": rec["clocks"], "gpu_launches": rec["gpu_launches"], "roofline": roofline,
           "profile_units": {"steps_run": args.steps + args.warmup, "ct_steps_per_step": rec["ct_steps_per_step"],
                             "slab_steps_per_step": rec["slab_steps_per_step"]}}
    if "e2e" in rec:
        out["e2e"] = rec["e2e"]

    if rank == 0 and world == 1 and not args.no_subrecords:
        sub = {}
        if args.workload != "config2":
            r2 = measure_dose("config2", args, 0, local_rank, 1, dev, 2, 3, with_e2e=True)
            k2 = rooflines(r2, "config2", hbm_gbs, sm_max_mhz, peak_kind)
            sub["config2"] = {k: r2[k] for k in ("workload", "value", "ms_per_step", "histories_per_plan", "plans_per_step", "e2e", "timing_ms_per_step", "gpu_launches")}
            sub["config2"]["e2e_over_value"] = r2["e2e"]["value"] / r2["value"]
            sub["config2"]["roofline"] = k2
        if args.workload != "config5_polygon":
            rp = measure_dose("config5_polygon", args, 0, local_rank, 1, dev, 2, 2, with_e2e=False)
            sub["config5_polygon"] = {k: rp[k] for k in ("workload", "value", "ms_per_step", "histories_per_plan", "timing_ms_per_step", "gpu_launches")}
            sub["config5_polygon"]["relative_to_bitmap"] = rp["value"] / rec["value"] if args.workload == "config5" else None
        sub["config3"] = measure_to_uncertainty(CONFIG3_SEEDS)
        sub["config4"] = measure_influence(10_000, 1, 1)
        out["configs"] = sub
        out["dose_at_0p5pct"] = {"workload": sub["config3"]["workload"], "seconds": sub["config3"]["seconds_mean"], "seconds_std": sub["config3"]["seconds_std"], "seconds_median": sub["config3"]["seconds_median"],
                                 "uncertainty_max": sub["config3"]["uncertainty_max"], "target": 0.005}
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import cpu_bench
        plans, n_default, _ = workload_plans(args.workload, args.plans)
        per_plan = args.cpu_sample // len(plans)
        busy, done, cores = 0.0, 0, 1
        for (_, fn, kw) in plans:
            r, cores, _ = cpu_bench.time_oracle(fn, kw, rec["histories_per_plan"], SEED, per_plan)
            busy += per_plan / r; done += per_plan
        out["cpu_baseline"] = {"value": done / busy, "unit": "histories/s", "cores": cores, "kind": "oracle",
                               "sample": "%d histories per plan over the %d plan(s), ids spread over the %d-history run, "
                                         "%d single-threaded oracle processes" % (per_plan, len(plans), rec["histories_per_plan"], cores)}
    if rank == 0:
        print(json.dumps(out))


def measure_to_uncertainty(seeds, target=0.005, batch=1_000_000):
    """Second half of the metric on configs[2]: per synthetic patient, seconds of set-up (vpmc_create + set_*
    from host arrays) + batches of 10^6 histories until the C6 estimator <= 0.5 %, the stopping rule evaluated on the device
    after every batch (vpmc_dose_to_uncertainty: one CUDA-graph WHILE node, no host round trip between batches)."""
    import numpy as np
    import torch
    from paper_2307_01416_b200 import binding, workloads as wl
    secs, hist, unc, reached = [], [], [], []
    for i, s in enumerate((seeds[0],) + tuple(seeds)):          # the first pass is an untimed warm-up (allocator cache, module load)
        p = wl.config3(s)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        e = binding.Engine(p)
        d = e.dose_to_uncertainty(batch, target, SEED, min_batches=2, max_batches=2000)
        nb, u, ok = e.run_info()
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        assert bool(torch.isfinite(d).all())
        e.close()
        if i > 0:
            secs.append(dt); hist.append(nb * batch); unc.append(u); reached.append(ok)
    a = np.asarray(secs)
    return {"workload": "BASELINE.json configs[2]: synthetic head CT 256x256x160 @ 1x1x1.5 mm, 2 beams with apertures, %d patients (seeds %d-%d), "
                        "each run to %.1f %% in batches of %d histories" % (len(seeds), seeds[0], seeds[-1], 100 * target, batch),
            "seconds": secs, "seconds_median": float(np.median(a)), "seconds_mean": float(a.mean()), "seconds_std": float(a.std(ddof=1)) if a.size > 1 else 0.0,
            "seconds_min": float(a.min()), "seconds_max": float(a.max()), "histories": hist, "uncertainty": unc,
            "uncertainty_max": float(max(unc)), "all_reached_target": bool(all(reached)),
            "paper_context": "VPMC 8.20 +- 6.42 s per plan on its 10 patients, 4 x NVIDIA Ampere (P:L187-198): other data, other hardware"}


def measure_influence(hps, steps, warmup):
    """configs[3]: the 13-scenario influence-matrix build (S7 + S8) on the config-3 head with ~2000 spots."""
    import torch
    from paper_2307_01416_b200 import binding, workloads as wl
    hbm_gbs, _, peak_kind = load_peaks()
    w = wl.config4(hist_per_spot=hps)
    eng = binding.Engine(w)
    sc = [binding.scenario(s, k) for s, k in w["scenarios"]]
    hps = int(hps)

    def step():
        res = eng.influence(sc, hps, w["rel_threshold"], SEED)
        nnz = sum(int(c.numel()) for (_, c, _) in res)
        fin = all(bool(torch.isfinite(v).all()) for (_, _, v) in res)
        del res
        return nnz, fin

    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    eng.set_timing(True); eng.timing()
    l0 = eng.launch_count()
    sampler = ClockSampler(torch.cuda.current_device()); sampler.start()
    t_ms = 0.0
    for _ in range(steps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        res = eng.influence(sc, hps, w["rel_threshold"], SEED)
        b.record(); torch.cuda.synchronize()
        t_ms += a.elapsed_time(b)
        nnz = sum(int(c.numel()) for (_, c, _) in res)
        assert all(bool(torch.isfinite(v).all()) for (_, _, v) in res), "non-finite CSR values"
        del res
    clocks = sampler.stop()
    tm = eng.timing()
    st = eng.influence_stats()
    opt = measure_optimiser(eng, sc, hps, w, hbm_gbs, peak_kind)
    tl = eng.tallies()                                                # of the last build: every history of every scenario once
    ct_steps = int(tl.as_dict()["n_steps_ct"])
    box = None
    vox_ms, vox_n = tm["voxel"][0] / steps, tm["voxel"][1] / steps
    if vox_ms > 0:
        _, sm_max_mhz, _ = load_peaks()
        peak = 148 * 4 * 32 * sm_max_mhz * 1e6 / 1e9
        counts = load_inst_counts("config4")
        row = counts.get("voxel_kernel_box") if counts else None
        ipu = float(row["thread_inst_per_unit"]) if row else None
        box = {"kernel": "voxel_kernel<1, ...> (BoxScorer)", "bound": "alu", "peak": peak, "unit": "Glane-inst/s", "ct_steps_per_build": ct_steps,
               "voxel_class_ms": vox_ms, "launches": vox_n, "inst_per_unit": ipu, "inst_per_unit_survey": SURVEY_INST_PER_STEP,
               "achieved": ipu * ct_steps / (vox_ms * 1e-3) / 1e9 if ipu else None,
               "frac": ipu * ct_steps / (vox_ms * 1e-3) / 1e9 / peak if ipu else None,
               "frac_survey_count": SURVEY_INST_PER_STEP * ct_steps / (vox_ms * 1e-3) / 1e9 / peak,
               "lanes_per_inst": float(row["lanes_per_inst"]) if row else None,
               "red": {"sectors_per_unit": float(row["red_sectors_per_unit"])} if row else None,
               "l2": {"bytes_per_unit": float(row["l2_bytes_per_unit"]), "hit_pct": float(row["l2_hit_pct"])} if row else None,
               "note": "the voxel timing class also holds the pilot launches (MODE 2, bounding boxes), whose steps are not counted: the fraction is a lower bound",
               "inst_source": "profiles/r2_inst_per_step.csv row (config4, voxel_kernel_box): ncu counters of the MODE 1 launches of a build at 2000 "
                              "histories per spot / CT steps counted by the kernels" if row else "no committed ncu counts for this config"}
    n_hist = len(sc) * eng.n_spots * hps
    wr_s = tm["writer"][0] * 1e-3 / steps
    alg = 8.0 * st["nnz"] + 12.0 * st["box_elements"]                 # nnz (col + val) written once + three 4-byte reads of every box element
    impl = 24.0 * st["nnz"] + 16.0 * st["box_elements"]               # + staging round trip of the rows, + the converted write-back
    out = {"value": n_hist * steps / (t_ms * 1e-3), "ms_per_step": t_ms / steps,
           "config": {"workload": "BASELINE.json configs[3]: 13-scenario influence matrices on the config-3 head (%s), %d spots, "
                                  "%d histories per spot, threshold 1e-4" % (w["name"], eng.n_spots, hps),
                      "l2_flush_between_steps": False, "inputs_larger_than_l2": True},
           "workload": "configs[3] influence build (%s, %d spots, %d histories per spot, 13 scenarios)" % (w["name"], eng.n_spots, hps),
           "seconds_per_13_matrices": t_ms * 1e-3 / steps, "nnz_total": nnz, "csr_bytes": nnz * 8 + 13 * (eng.n_spots + 1) * 8,
           "clocks": clocks, "gpu_launches": eng.launch_count() - l0, "stats": st,
           "timing_ms_per_step": {k: v[0] / steps for k, v in tm.items()},
           "share_of_step": {k: v[0] / t_ms for k, v in tm.items()},
           "writer": {"bound": "hbm", "seconds": wr_s, "algorithmic_bytes": alg, "achieved": alg / wr_s / 1e9 if wr_s > 0 else None, "peak": hbm_gbs,
                      "unit": "GB/s", "frac": alg / wr_s / 1e9 / hbm_gbs if wr_s > 0 else None,
                      "bytes_as_implemented": impl, "achieved_as_implemented": impl / wr_s / 1e9 if wr_s > 0 else None,
                      "note": "algorithmic = 8 B x nnz written + 3 reads x 4 B of every box element (max, count, emit); the class also times the "
                              "overflow-list kernels", "peak_source": peak_kind + " MEASURED_PEAKS.json hbm_gbs"},
           "optimiser_iteration": opt, "roofline_voxel_box": box,
           "profile_units": {"builds_run": warmup + steps + 1, "ct_steps_per_build": ct_steps},
           "paper_context": "41.6 s for 13 influence matrices (P:L205-207): other data, other hardware"}
    eng.close()
    return out


def measure_optimiser(eng, sc, hps, w, hbm_gbs, peak_kind, iters=5):
    """SURVEY.md 8(f)-1 on the matrices just built: seconds per robust-optimiser iteration (13 dose products, the voxel-wise
    worst case, 13 gradient products) with the 13 matrices resident in HBM; every entry streams through twice."""
    import torch
    mats = eng.influence(sc, hps, w["rel_threshold"], SEED)
    nnz = sum(int(c.numel()) for (_, c, _) in mats)
    n_sc, nvox = len(mats), eng.nvox
    wts = torch.full((eng.n_spots,), 1.0e8, dtype=torch.float32, device="cuda")
    d0 = eng.spmv_dose(mats[0], wts)
    target = (0.95 * d0).contiguous()
    weight = (d0 > 0.05 * d0.max()).float()
    ws = (torch.empty((n_sc, nvox), dtype=torch.float32, device="cuda"), torch.empty((n_sc, nvox), dtype=torch.float32, device="cuda"))
    obj, grad, _ = eng.robust_iteration(mats, wts, target, weight, ws=ws)          # warm-up
    torch.cuda.synchronize()
    assert bool(torch.isfinite(grad).all())
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")
    t_ms = 0.0
    for _ in range(iters):
        flush.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        obj, grad, _ = eng.robust_iteration(mats, wts, target, weight, ws=ws)
        b.record(); torch.cuda.synchronize()
        t_ms += a.elapsed_time(b)
    sec = t_ms * 1e-3 / iters
    alg = 16.0 * nnz + 4.0 * 4.0 * n_sc * nvox       # every entry (col + val) read twice; per scenario the dose and residual vectors written and read once each
    del mats
    return {"seconds_per_iteration": sec, "nnz": nnz, "scenarios": n_sc, "bound": "hbm", "algorithmic_bytes": alg, "achieved": alg / sec / 1e9,
            "peak": hbm_gbs, "unit": "GB/s", "frac": alg / sec / 1e9 / hbm_gbs, "objective": float(obj), "peak_source": peak_kind + " MEASURED_PEAKS.json hbm_gbs",
            "l2_flush_between_iterations": True,
            "paper_context": "0.1-0.3 s per iteration on 4 x A100 (P:L95): other data, other hardware"}


if __name__ == "__main__":
    main()
