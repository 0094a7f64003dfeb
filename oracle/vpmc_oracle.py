"""ctypes face of the CPU oracle (oracle/vpmc_oracle.c).  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It imports nothing from the CUDA package
(paper_2307_01416_b200); problems are described with plain numpy arrays / dicts as
produced by the seeded workload generators.

The C file is the oracle; this module only marshals arguments, plus two numpy
estimators that SURVEY.md 8(c)-C6 defines on top of the transport result (batch
uncertainty, 3D gamma).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "vpmc_oracle.c")
_LIB = os.path.join(_HERE, "libvpmc_oracle.so")

FLAG_MCS, FLAG_STRAGGLE, FLAG_NUCLEAR = 1, 2, 4
REG_VAC, REG_RS, REG_AP_OPEN, REG_AP_BRASS, REG_CT = 0, 1, 2, 3, 4
CONT, STOPPED, NUCLEAR, ESCAPED = 0, 1, 2, 3


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, no fast-math: fp64 semantics as written)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fno-fast-math",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class Params(C.Structure):
    _fields_ = [(n, C.c_double) for n in (
        "alpha", "p", "X0_w", "Es", "c_log", "beta_nuc", "gamma_loc", "k_bohr", "za_w",
        "R_cut", "f_R", "s_max", "s_rs", "s_ap",
        "brass_rsp", "brass_rho", "brass_X0", "brass_za",
        "rs_rsp", "rs_rho", "rs_X0", "rho_min", "delta_E")] + [("flags", C.c_int32), ("n_batches", C.c_int32)]


def default_params(**kw) -> Params:
    """SURVEY.md 8(c)-C0 defaults."""
    p = Params(alpha=0.022, p=1.77, X0_w=360.8, Es=13.6, c_log=0.038, beta_nuc=0.0012, gamma_loc=0.6,
               k_bohr=0.015692, za_w=0.5551, R_cut=0.1, f_R=0.25, s_max=float("inf"), s_rs=1.0, s_ap=1.0,
               brass_rsp=5.523, brass_rho=8.5, brass_X0=14.94, brass_za=0.457,
               rs_rsp=1.0, rs_rho=1.0, rs_X0=360.8, rho_min=1e-3, delta_E=0.0,
               flags=FLAG_MCS | FLAG_STRAGGLE | FLAG_NUCLEAR, n_batches=10)
    for k, v in kw.items():
        if not hasattr(p, k):
            raise KeyError(k)
        setattr(p, k, v)
    return p


def params_as_f32(p: Params) -> Params:
    """Round every real parameter to the nearest fp32 value (what the C-ABI struct holds)."""
    q = Params()
    for name, typ in Params._fields_:
        v = getattr(p, name)
        setattr(q, name, float(np.float32(v)) if typ is C.c_double else v)
    return q


class _Ct(C.Structure):
    _fields_ = [("n", C.c_int32 * 3), ("h", C.c_double * 3), ("origin", C.c_double * 3), ("hu", C.c_void_p)]


class _Calib(C.Structure):
    _fields_ = [("n", C.c_int32), ("hu", C.c_void_p), ("rsp", C.c_void_p), ("rho", C.c_void_p), ("xsp", C.c_void_p)]


class _Beam(C.Structure):
    _fields_ = [("iso", C.c_double * 3), ("rot", C.c_double * 9), ("n_spots", C.c_int32),
                ("x", C.c_void_p), ("y", C.c_void_p), ("E", C.c_void_p), ("w", C.c_void_p), ("sigma", C.c_void_p),
                ("rs_wet", C.c_double), ("rs_face", C.c_double), ("ap_present", C.c_int32),
                ("ap_T", C.c_double), ("ap_face", C.c_double), ("ap_open", C.c_void_p),
                ("ap_nx", C.c_int32), ("ap_ny", C.c_int32),
                ("ap_u0", C.c_double), ("ap_v0", C.c_double), ("ap_du", C.c_double), ("ap_dv", C.c_double),
                ("ap_n_poly", C.c_int32), ("ap_poly", C.c_void_p)]


class _Problem(C.Structure):
    _fields_ = [("P", Params), ("ct", _Ct), ("cal", _Calib), ("n_beams", C.c_int32), ("beams", C.c_void_p)]


class Scenario(C.Structure):
    _fields_ = [("shift", C.c_double * 3), ("rsp_scale", C.c_double)]


class Tallies(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("incident", "dep_ct", "dep_rs", "dep_brass", "escaped", "removed")] + \
               [(n, C.c_uint64) for n in ("n_stopped_ct", "n_stopped_rs", "n_stopped_brass", "n_nuclear", "n_escaped")]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


class StepRec(C.Structure):
    _fields_ = [("hid", C.c_uint64), ("step", C.c_int32), ("region", C.c_int32), ("cause", C.c_int32),
                ("ivox", C.c_int32 * 3), ("r", C.c_double * 3), ("u", C.c_double * 3),
                ("E_before", C.c_double), ("E_after", C.c_double), ("s", C.c_double),
                ("t_rad", C.c_double), ("tau", C.c_double), ("tau_star", C.c_double), ("dep", C.c_double)]


STEP_DTYPE = np.dtype([("hid", "<u8"), ("step", "<i4"), ("region", "<i4"), ("cause", "<i4"), ("ivox", "<i4", 3),
                       ("r", "<f8", 3), ("u", "<f8", 3), ("E_before", "<f8"), ("E_after", "<f8"), ("s", "<f8"),
                       ("t_rad", "<f8"), ("tau", "<f8"), ("tau_star", "<f8"), ("dep", "<f8")],
                      align=True)

DIGEST_DTYPE = np.dtype([("hid", "<u8"), ("hash", "<u8"), ("n_rec", "<i4"), ("cause", "<i4"), ("r", "<f8", 3),
                         ("E_last", "<f8"), ("dep_ct", "<f8")], align=True)

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        sizes = (C.c_int32 * 8)()
        _lib.orc_sizes(sizes)
        mine = [C.sizeof(t) for t in (Params, _Ct, _Calib, _Beam, _Problem, Scenario, Tallies, StepRec)]
        assert list(sizes) == mine, (list(sizes), mine)
        assert STEP_DTYPE.itemsize == C.sizeof(StepRec)
        _lib.orc_u01.restype = C.c_double
        _lib.orc_u01.argtypes = [C.c_uint32]
        _lib.orc_csr_row.restype = C.c_int64
        _lib.orc_csr_row.argtypes = [C.c_void_p, C.c_int64, C.c_float, C.c_void_p, C.c_void_p]
    return _lib


def scenario(shift=(0.0, 0.0, 0.0), rsp_scale=1.0) -> Scenario:
    s = Scenario()
    s.shift[:] = [float(x) for x in shift]
    s.rsp_scale = float(rsp_scale)
    return s


def _f64(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


@dataclass
class Problem:
    """A transport problem in the oracle's own (fp64) terms, built from plain arrays.

    ct: dict(n=(nx,ny,nz), h=(hx,hy,hz), origin=(ox,oy,oz), hu=int16[nz,ny,nx] or flat)
    calib: dict(hu=[], rsp=[], rho=[], xsp=None|[])
    beams: list of dict(iso, rot(3x3), spots=float array [n,5] = x,y,E,w,sigma,
                        rs_wet=0, rs_face=190, aperture=None|dict(T, face, open=uint8[ny,nx], u0, v0, du, dv))
    """
    ct: dict
    calib: dict
    beams: list
    params: Params = field(default_factory=default_params)
    _keep: list = field(default_factory=list, repr=False)
    _c: _Problem | None = field(default=None, repr=False)

    def cstruct(self) -> _Problem:
        if self._c is not None:
            return self._c
        keep = self._keep
        pb = _Problem()
        pb.P = self.params
        hu = np.ascontiguousarray(np.asarray(self.ct["hu"], dtype=np.int16).reshape(-1))
        keep.append(hu)
        n = [int(x) for x in self.ct["n"]]
        assert hu.size == n[0] * n[1] * n[2]
        pb.ct.n[:] = n
        pb.ct.h[:] = [float(x) for x in self.ct["h"]]
        pb.ct.origin[:] = [float(x) for x in self.ct["origin"]]
        pb.ct.hu = hu.ctypes.data
        cal = {k: (None if self.calib.get(k) is None else _f64(self.calib[k])) for k in ("hu", "rsp", "rho", "xsp")}
        keep.append(cal)
        pb.cal.n = int(cal["hu"].size)
        pb.cal.hu, pb.cal.rsp, pb.cal.rho = cal["hu"].ctypes.data, cal["rsp"].ctypes.data, cal["rho"].ctypes.data
        pb.cal.xsp = None if cal["xsp"] is None else cal["xsp"].ctypes.data
        arr = (_Beam * len(self.beams))()
        for i, b in enumerate(self.beams):
            sp = _f64(b["spots"]).reshape(-1, 5)
            cols = [np.ascontiguousarray(sp[:, k]) for k in range(5)]
            keep.append(cols)
            arr[i].iso[:] = [float(x) for x in b["iso"]]
            arr[i].rot[:] = [float(x) for x in np.asarray(b["rot"], dtype=np.float64).reshape(9)]
            arr[i].n_spots = sp.shape[0]
            arr[i].x, arr[i].y, arr[i].E, arr[i].w, arr[i].sigma = [c.ctypes.data for c in cols]
            arr[i].rs_wet = float(b.get("rs_wet", 0.0))
            arr[i].rs_face = float(b.get("rs_face", 190.0))
            ap = b.get("aperture")
            arr[i].ap_present = 0 if ap is None else 1
            if ap is not None and ap.get("polygon") is not None:      # polygon opening, no bitmap
                poly = _f64(ap["polygon"]).reshape(-1, 2)
                keep.append(poly)
                arr[i].ap_T, arr[i].ap_face = float(ap["T"]), float(ap.get("face", 150.0))
                arr[i].ap_n_poly, arr[i].ap_poly = poly.shape[0], poly.ctypes.data
            elif ap is not None:
                op = np.ascontiguousarray(np.asarray(ap["open"], dtype=np.uint8))
                keep.append(op)
                arr[i].ap_T, arr[i].ap_face = float(ap["T"]), float(ap.get("face", 150.0))
                arr[i].ap_open = op.ctypes.data
                arr[i].ap_ny, arr[i].ap_nx = op.shape
                arr[i].ap_u0, arr[i].ap_v0 = float(ap["u0"]), float(ap["v0"])
                arr[i].ap_du, arr[i].ap_dv = float(ap["du"]), float(ap["dv"])
        keep.append(arr)
        pb.n_beams = len(self.beams)
        pb.beams = C.addressof(arr)
        self._c = pb
        return pb

    @property
    def nvox(self) -> int:
        n = self.ct["n"]
        return int(n[0]) * int(n[1]) * int(n[2])

    @property
    def n_spots(self) -> int:
        return sum(np.asarray(b["spots"]).reshape(-1, 5).shape[0] for b in self.beams)

    @property
    def total_weight(self) -> float:
        """W = sum of spot weights in index order, fp64 (C2)."""
        W = 0.0
        for b in self.beams:
            for w in _f64(b["spots"]).reshape(-1, 5)[:, 3]:
                W += float(w)
        return W


# ----------------------------------------------------------------------------- calls

def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) & 0xFFFFFFFF for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) & 0xFFFFFFFF for x in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def u01(x: int) -> float:
    return float(lib().orc_u01(C.c_uint32(int(x) & 0xFFFFFFFF)))


def apportion(N: int, w) -> np.ndarray:
    w = _f64(w)
    out = np.zeros(w.size, dtype=np.uint64)
    lib().orc_apportion(C.c_uint64(int(N)), C.c_void_p(w.ctypes.data), C.c_int32(w.size), C.c_void_p(out.ctypes.data))
    return out


def calib_eval(calib: dict, hu: float):
    cal = _Calib()
    arrs = {k: (None if calib.get(k) is None else _f64(calib[k])) for k in ("hu", "rsp", "rho", "xsp")}
    cal.n = int(arrs["hu"].size)
    cal.hu, cal.rsp, cal.rho = arrs["hu"].ctypes.data, arrs["rsp"].ctypes.data, arrs["rho"].ctypes.data
    cal.xsp = None if arrs["xsp"] is None else arrs["xsp"].ctypes.data
    out = (C.c_double * 3)()
    lib().orc_calib_eval(C.byref(cal), C.c_double(float(hu)), out)
    return tuple(out)


def point_in_polygon(poly, x: float, y: float) -> bool:
    """The oracle's crossing-number test (ref. 67) of point (x, y) against the closed polygon poly [n, 2]."""
    p = _f64(poly).reshape(-1, 2)
    lib().orc_point_in_polygon.restype = C.c_int
    return bool(lib().orc_point_in_polygon(C.c_void_p(p.ctypes.data), C.c_int32(p.shape[0]), C.c_double(float(x)), C.c_double(float(y))))


def spot_counts(pb: Problem, N: int) -> np.ndarray:
    out = np.zeros(pb.n_spots, dtype=np.uint64)
    lib().orc_spot_counts(C.byref(pb.cstruct()), C.c_uint64(int(N)), C.c_void_p(out.ctypes.data))
    return out


def dose_edep(pb: Problem, N: int, seed: int, sc: Scenario | None = None, hid_begin: int = 0,
              hid_end: int | None = None, batch: int = 0, n_batches: int = 1, edep: np.ndarray | None = None,
              hid_offset: int = 0):
    """E_dep [MeV] (fp64, flat nvox) of history ids [hid_begin, hid_end) of an N-history dose run; hid_offset is added
    to every id before it keys the random stream (sequential batches, R15)."""
    sc = sc or scenario()
    if edep is None:
        edep = np.zeros(pb.nvox, dtype=np.float64)
    tal = Tallies()
    rc = lib().orc_dose_edep_offset(C.byref(pb.cstruct()), C.byref(sc), C.c_uint64(int(N)), C.c_uint64(int(seed)),
                                    C.c_uint64(int(hid_begin)), C.c_uint64(int(N if hid_end is None else hid_end)),
                                    C.c_int32(batch), C.c_int32(n_batches), C.c_uint64(int(hid_offset)),
                                    C.c_void_p(edep.ctypes.data), C.byref(tal))
    assert rc == 0
    return edep, tal


def dose_from_edep(pb: Problem, edep: np.ndarray, scale: float) -> np.ndarray:
    out = np.zeros(pb.nvox, dtype=np.float64)
    e = _f64(edep)
    lib().orc_dose_from_edep(C.byref(pb.cstruct()), C.c_void_p(e.ctypes.data), C.c_double(float(scale)),
                             C.c_void_p(out.ctypes.data))
    return out


def coarse_cells(pb: Problem, div):
    """SURVEY 8(f)-4 / include/vpmc.h vpmc_set_scoring_grid: cell index of every voxel (flat, v = ix + nx (iy + ny iz)) for cells of
    div voxels per axis, and the scoring grid's dimensions sn = ceil(n / div); cell c = cx + sn_x (cy + sn_y cz)."""
    n = [int(x) for x in pb.ct["n"]]
    sn = [(n[a] + int(div[a]) - 1) // int(div[a]) for a in range(3)]
    iz, iy, ix = np.meshgrid(np.arange(n[2]) // int(div[2]), np.arange(n[1]) // int(div[1]), np.arange(n[0]) // int(div[0]), indexing="ij")
    return (ix + sn[0] * (iy + sn[1] * iz)).reshape(-1), sn


def dose_from_edep_coarse(pb: Problem, edep: np.ndarray, scale: float, div) -> np.ndarray:
    """Dose of the scoring cells: energy of a cell / mass of a cell, the density floored per voxel as in C6:
    dose[c] = scale * sum_{v in c} E_dep[v] / (V_vox * sum_{v in c} max(rho_v, rho_min)) * 1.602176634e-10 Gy."""
    cell, sn = coarse_cells(pb, div)
    ncell = sn[0] * sn[1] * sn[2]
    hu = np.asarray(pb.ct["hu"], dtype=np.float64).reshape(-1)
    rho = np.interp(hu, _f64(pb.calib["hu"]), _f64(pb.calib["rho"]))          # piecewise linear, clamped at the end nodes (C5)
    rho = np.maximum(rho, float(pb.params.rho_min))
    h = [float(x) for x in pb.ct["h"]]
    V = h[0] * h[1] * h[2] * 1e-3
    e_c = np.bincount(cell, weights=_f64(edep), minlength=ncell)
    m_c = np.bincount(cell, weights=rho, minlength=ncell) * V
    return float(scale) * e_c / m_c * 1.602176634e-10


def dose(pb: Problem, N: int, seed: int, sc: Scenario | None = None):
    """Full dose-mode result: dose [Gy] (fp64, flat), tallies.  scale = W/N (C6)."""
    e, tal = dose_edep(pb, N, seed, sc)
    return dose_from_edep(pb, e, pb.total_weight / float(N)), tal


def influence_edep(pb: Problem, g: int, hist_per_spot: int, seed: int, sc: Scenario | None = None,
                   i_begin: int = 0, i_end: int | None = None, edep: np.ndarray | None = None):
    sc = sc or scenario()
    if edep is None:
        edep = np.zeros(pb.nvox, dtype=np.float64)
    tal = Tallies()
    rc = lib().orc_influence_edep(C.byref(pb.cstruct()), C.byref(sc), C.c_int32(int(g)), C.c_uint32(int(hist_per_spot)),
                                  C.c_uint64(int(seed)), C.c_uint32(int(i_begin)),
                                  C.c_uint32(int(hist_per_spot if i_end is None else i_end)),
                                  C.c_void_p(edep.ctypes.data), C.byref(tal))
    assert rc == 0
    return edep, tal


def influence_column(pb: Problem, g: int, hist_per_spot: int, seed: int, sc: Scenario | None = None) -> np.ndarray:
    """Dense fp32 influence column of global spot g (Gy per unit spot weight), scale 1/hist_per_spot (C6)."""
    e, _ = influence_edep(pb, g, hist_per_spot, seed, sc)
    return dose_from_edep(pb, e, 1.0 / float(hist_per_spot)).astype(np.float32)


def csr_row(col: np.ndarray, rel_thr: float):
    col = np.ascontiguousarray(col, dtype=np.float32)
    n = lib().orc_csr_row(C.c_void_p(col.ctypes.data), C.c_int64(col.size), C.c_float(rel_thr), None, None)
    idx = np.zeros(n, dtype=np.int32)
    val = np.zeros(n, dtype=np.float32)
    lib().orc_csr_row(C.c_void_p(col.ctypes.data), C.c_int64(col.size), C.c_float(rel_thr),
                      C.c_void_p(idx.ctypes.data), C.c_void_p(val.ctypes.data))
    return idx, val


def influence_csr(pb: Problem, hist_per_spot: int, rel_thr: float, seed: int, sc: Scenario | None = None,
                  spots=None):
    """CSR (row_ptr int64, col int32, val fp32) of one scenario, rows = spots in input order (C6)."""
    spots = range(pb.n_spots) if spots is None else spots
    row_ptr, cols, vals = [0], [], []
    for g in spots:
        i, v = csr_row(influence_column(pb, g, hist_per_spot, seed, sc), rel_thr)
        cols.append(i)
        vals.append(v)
        row_ptr.append(row_ptr[-1] + i.size)
    return (np.asarray(row_ptr, dtype=np.int64),
            np.concatenate(cols) if cols else np.zeros(0, np.int32),
            np.concatenate(vals) if vals else np.zeros(0, np.float32))


def trace(pb: Problem, hids, n_or_hps: int, seed: int, sc: Scenario | None = None, mode: int = 0,
          max_steps: int = 1024):
    """Per-history numpy record arrays (STEP_DTYPE) of the selected history ids."""
    sc = sc or scenario()
    hids = np.ascontiguousarray(np.asarray(hids, dtype=np.uint64))
    recs = np.zeros((hids.size, max_steps), dtype=STEP_DTYPE)
    nrec = np.zeros(hids.size, dtype=np.int32)
    rc = lib().orc_trace(C.byref(pb.cstruct()), C.byref(sc), C.c_int32(mode), C.c_uint64(int(n_or_hps)),
                         C.c_uint64(int(seed)), C.c_void_p(hids.ctypes.data), C.c_int32(hids.size),
                         C.c_int32(max_steps), C.c_void_p(recs.ctypes.data), C.c_void_p(nrec.ctypes.data))
    assert rc == 0
    assert (nrec <= max_steps).all(), "max_steps too small"
    return [recs[i, :nrec[i]] for i in range(hids.size)]


def digests(pb: Problem, N: int, seed: int, hid_begin: int, n: int, sc: Scenario | None = None) -> np.ndarray:
    """DIGEST_DTYPE array of history ids [hid_begin, hid_begin + n) of the N-history dose run."""
    sc = sc or scenario()
    out = np.zeros(n, dtype=DIGEST_DTYPE)
    rc = lib().orc_digests(C.byref(pb.cstruct()), C.byref(sc), C.c_uint64(int(N)), C.c_uint64(int(seed)),
                           C.c_uint64(int(hid_begin)), C.c_int32(int(n)), C.c_void_p(out.ctypes.data))
    assert rc == 0
    return out


class injected_uniforms:
    """Context manager of the oracle's test hook: the transport block (purpose 0) of step k is u[k] (4 numbers)
    for k < len(u); later steps draw from Philox as usual."""

    def __init__(self, u):
        self.u = np.ascontiguousarray(np.asarray(u, dtype=np.float64).reshape(-1, 4))

    def __enter__(self):
        lib().orc_inject_uniforms(C.c_void_p(self.u.ctypes.data), C.c_int32(self.u.shape[0]))
        return self

    def __exit__(self, *exc):
        lib().orc_inject_uniforms(None, C.c_int32(0))
        return False


# ----------------------------------------------------------------------------- C6 estimators (numpy)

def batch_uncertainty(batch_doses: np.ndarray) -> float:
    """C6: batch_doses [B, nvox], each scaled to full weight.  sigma_v^2 = sum_b (D_b - Dbar)^2 / (B(B-1));
    returns mean of sigma_v / Dbar_v over voxels with Dbar_v >= 0.5 max Dbar."""
    D = np.asarray(batch_doses, dtype=np.float64)
    B = D.shape[0]
    mean = D.mean(axis=0)
    var = ((D - mean) ** 2).sum(axis=0) / (B * (B - 1))
    sel = mean >= 0.5 * mean.max()
    return float(np.mean(np.sqrt(var[sel]) / mean[sel]))


def dose_to_uncertainty(pb: Problem, batch_histories: int, target: float, seed: int, min_batches: int = 2,
                        max_batches: int = 1000, sc: Scenario | None = None):
    """SURVEY.md 8(d) metric (2) / P:L107, "<0.5 %": sequential stopping rule.  Batches of `batch_histories`
    histories are run one after another -- the k-th (k = 0, 1, ...) is the batch_histories-history plan sample with
    history ids k 2^32 + i (R15) -- and after each the C6 estimator over the batch doses so far is
    evaluated; stop as soon as k + 1 >= min_batches and the estimate <= target (or at max_batches).
    Returns (dose [Gy], batches used, list of the estimates after each batch from the second on)."""
    batches, history = [], []
    scale = pb.total_weight / float(batch_histories)
    while len(batches) < max_batches:
        k = len(batches)
        e, _ = dose_edep(pb, batch_histories, seed, sc, hid_offset=k << 32)
        batches.append(dose_from_edep(pb, e, scale))
        if len(batches) >= 2:
            history.append(batch_uncertainty(np.array(batches)))
            if len(batches) >= min_batches and history[-1] <= target:
                break
    return np.mean(np.array(batches), axis=0), len(batches), history


def gamma_counts(ref: np.ndarray, ev: np.ndarray, h, dd: float = 0.01, dta: float = 1.0, thr: float = 0.1, sub: int = 10):
    """C6 / P:L107: global 3D gamma.  ref, ev: [nz, ny, nx]; h = (hx, hy, hz) mm; dd relative to the reference
    maximum; voxels with ref >= thr*max evaluated; pass iff gamma <= 1.  Zero-distance test first, full search
    with trilinear sub-sampling at h/sub only for voxels failing it.  Returns (voxels evaluated, voxels failing)."""
    from scipy.ndimage import map_coordinates
    ref = np.asarray(ref, dtype=np.float64)
    ev = np.asarray(ev, dtype=np.float64)
    mx = ref.max()
    dcrit = dd * mx
    sel = ref >= thr * mx
    n_eval = int(sel.sum())
    if n_eval == 0:
        return 0, 0
    fail = sel & (np.abs(ev - ref) > dcrit)
    idx = np.argwhere(fail)
    if idx.size == 0:
        return n_eval, 0
    hz, hy, hx = float(h[2]), float(h[1]), float(h[0])
    rng = [np.arange(-int(np.ceil(dta / s * sub)), int(np.ceil(dta / s * sub)) + 1) / sub for s in (hz, hy, hx)]
    oz, oy, ox = np.meshgrid(*rng, indexing="ij")
    dist2 = ((oz * hz) ** 2 + (oy * hy) ** 2 + (ox * hx) ** 2) / dta ** 2
    keep = dist2 <= 1.0
    oz, oy, ox, dist2 = oz[keep], oy[keep], ox[keep], dist2[keep]
    n_fail = 0
    for (z, y, x) in idx:
        vals = map_coordinates(ev, [z + oz, y + oy, x + ox], order=1, mode="nearest")
        g2 = dist2 + ((vals - ref[z, y, x]) / dcrit) ** 2
        if g2.min() > 1.0:
            n_fail += 1
    return n_eval, n_fail


def gamma_pass_rate(ref: np.ndarray, ev: np.ndarray, h, dd: float = 0.01, dta: float = 1.0, thr: float = 0.1,
                    sub: int = 10) -> float:
    """Pass rate 1 - failing / evaluated of gamma_counts (1.0 when no voxel is evaluated)."""
    n_eval, n_fail = gamma_counts(ref, ev, h, dd, dta, thr, sub)
    return 1.0 if n_eval == 0 else 1.0 - n_fail / n_eval
