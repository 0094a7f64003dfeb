"""Timing harness of the CPU oracle for bench.py's cpu_baseline / --impl reference legs.  TEST INFRASTRUCTURE.

The oracle stays single-threaded; all host cores are used by running independent processes on disjoint history-id
ranges (legal because streams are keyed by history id)."""
from __future__ import annotations

import os
import time


def _worker(args):
    wl_name, wl_kwargs, N, seed, lo, hi = args
    import numpy as np  # noqa: F401
    from oracle import vpmc_oracle as orc
    from paper_2307_01416_b200 import workloads
    w = getattr(workloads, wl_name)(**wl_kwargs)
    pb = orc.Problem(ct=w["ct"], calib=w["calib"], beams=w["beams"], params=orc.params_as_f32(orc.default_params()))
    t0 = time.perf_counter()
    e, tal = orc.dose_edep(pb, N, seed, hid_begin=lo, hid_end=hi)
    return time.perf_counter() - t0, float(e.sum()), hi - lo


def n_cores() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def time_oracle(wl_name: str, wl_kwargs: dict, N: int, seed: int, sample: int, cores: int | None = None):
    """Transport `sample` histories (ids spread over the whole N-history run in `cores` equal slices) of workload
    wl_name; returns (histories per second over all cores, cores used, wall seconds)."""
    import multiprocessing as mp
    from oracle import vpmc_oracle as orc
    orc.build()
    cores = cores or n_cores()
    per = max(sample // cores, 1)
    stride = N // cores
    jobs = [(wl_name, wl_kwargs, N, seed, k * stride, min(k * stride + per, N)) for k in range(cores)]
    ctx = mp.get_context("spawn")
    t0 = time.perf_counter()
    with ctx.Pool(cores) as pool:
        res = pool.map(_worker, jobs)
    wall = time.perf_counter() - t0
    busy = max(r[0] for r in res)
    done = sum(r[2] for r in res)
    return done / busy, cores, wall
