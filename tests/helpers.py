"""Shared test helpers: workload dict -> oracle Problem, and small utilities."""
import numpy as np

from oracle import vpmc_oracle as orc


def oracle_problem(wl: dict, params=None, f32_params=True) -> orc.Problem:
    p = params if params is not None else orc.default_params()
    if f32_params:
        p = orc.params_as_f32(p)
    return orc.Problem(ct=wl["ct"], calib=wl["calib"], beams=wl["beams"], params=p)


def grid(wl, flat):
    n = wl["ct"]["n"]
    return np.asarray(flat).reshape(n[2], n[1], n[0])


def read_golden(name):
    """Whitespace-separated rows, '#' comments."""
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", name)
    rows = []
    with open(path) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if line:
                rows.append(line.split())
    return rows
