"""ctypes face of robust_oracle.c -- TEST INFRASTRUCTURE (see the C file's header).  One iteration of the voxel-wise
worst-case robust optimiser on CSR influence matrices (R16), fp64."""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(_HERE, "robust_oracle.c")
LIB = os.path.join(_HERE, "librobust_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < os.path.getmtime(SRC):
        tmp = LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-o", tmp, SRC])
        os.replace(tmp, LIB)
    return LIB


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orb_worst_case.restype = C.c_double
        _lib = L
    return _lib


def _p(a):
    return C.c_void_p(a.ctypes.data)


def _csr(m):
    rp, col, val = m
    return (np.ascontiguousarray(rp, dtype=np.int64), np.ascontiguousarray(col, dtype=np.int32),
            np.ascontiguousarray(val, dtype=np.float32))


def spmv_dose(m, n_cols: int, w) -> np.ndarray:
    rp, col, val = _csr(m)
    w = np.ascontiguousarray(w, dtype=np.float64)
    d = np.zeros(n_cols, dtype=np.float64)
    lib().orb_spmv_dose(_p(rp), _p(col), _p(val), C.c_int32(rp.size - 1), C.c_int64(n_cols), _p(w), _p(d))
    return d


def spmv_grad(m, r, g=None) -> np.ndarray:
    rp, col, val = _csr(m)
    r = np.ascontiguousarray(r, dtype=np.float64)
    acc = g is not None
    if g is None:
        g = np.zeros(rp.size - 1, dtype=np.float64)
    lib().orb_spmv_grad(_p(rp), _p(col), _p(val), C.c_int32(rp.size - 1), _p(r), C.c_int32(1 if acc else 0), _p(g))
    return g


def worst_case(doses, target, weight):
    """(f, resid [n_sc, n], worst [n]) of the voxel-wise worst case."""
    doses = np.ascontiguousarray(doses, dtype=np.float64)
    n_sc, n = doses.shape
    t = np.ascontiguousarray(target, dtype=np.float64)
    p = np.ascontiguousarray(weight, dtype=np.float64)
    resid = np.zeros_like(doses)
    worst = np.zeros(n, dtype=np.int32)
    f = lib().orb_worst_case(_p(doses), C.c_int32(n_sc), C.c_int64(n), _p(t), _p(p), _p(resid), _p(worst))
    return float(f), resid, worst


def iteration(mats, n_cols: int, w, target, weight):
    """One iteration: (f, gradient [n_rows], doses [n_sc, n_cols])."""
    doses = np.stack([spmv_dose(m, n_cols, w) for m in mats])
    f, resid, _ = worst_case(doses, target, weight)
    g = None
    for s, m in enumerate(mats):
        g = spmv_grad(m, resid[s], g) if g is not None else spmv_grad(m, resid[s])
    return f, g, doses
