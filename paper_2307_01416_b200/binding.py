"""Thin ctypes binding of libvpmc.so (include/vpmc.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C-ABI.  PyTorch is used for device buffers and
streams.  There is no CPU fallback: if the library is missing or there is no CUDA device, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("VPMC_LIB", os.path.join(_HERE, "libvpmc.so"))   # VPMC_LIB: another build of the same library

OK, ERR_INVALID_ARG, ERR_GEOMETRY, ERR_CUDA, ERR_ALLOC, ERR_STATE = 0, -1, -2, -3, -4, -5
FLAG_MCS, FLAG_STRAGGLE, FLAG_NUCLEAR = 1, 2, 4
BRASS = 1

EXPORTS = ["vpmc_version", "vpmc_default_params", "vpmc_create", "vpmc_destroy", "vpmc_add_beam", "vpmc_set_beam",
           "vpmc_set_range_shifter", "vpmc_set_aperture", "vpmc_dose", "vpmc_dose_scenario", "vpmc_dose_host",
           "vpmc_set_history_window", "vpmc_influence", "vpmc_csr_from_dense", "vpmc_get_tallies",
           "vpmc_get_uncertainty", "vpmc_trace", "vpmc_get_launch_count", "vpmc_last_error", "vpmc_set_timing",
           "vpmc_get_timing", "vpmc_set_workspace_limit", "vpmc_step_from_state", "vpmc_set_knob", "vpmc_digests", "vpmc_dose_to_uncertainty",
           "vpmc_get_run_info", "vpmc_bench_red", "vpmc_get_aperture_tables", "vpmc_set_shard", "vpmc_get_influence_stats", "vpmc_spmv_dose", "vpmc_spmv_grad",
           "vpmc_worst_case", "vpmc_robust_iteration", "vpmc_spmv_grad_static", "vpmc_set_aperture_polygon", "vpmc_gamma", "vpmc_set_scoring_grid",
           "vpmc_get_scoring_dims"]

STEP_SOURCE, STEP_DRIFT_TO_RS, STEP_RS, STEP_DRIFT_TO_AP, STEP_AP, STEP_CT_ENTRY, STEP_CT = range(7)
STATIC_MAX_NNZ = 1 << 28          # VPMC_STATIC_MAX_NNZ
KNOB_CHUNK, KNOB_BOX_GROW, KNOB_BOX_PAD, KNOB_OVF_CAP, KNOB_LUT_GLOBAL, KNOB_VERBOSE, KNOB_OVF_SORT_CAP = range(7)


class VpmcError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("vpmc error %d: %s" % (code, msg))
        self.code = code


class Params(C.Structure):
    _fields_ = [(n, C.c_float) for n in (
        "alpha", "p", "X0_w", "Es", "c_log", "beta_nuc", "gamma_loc", "k_bohr", "za_w", "R_cut", "f_R", "s_max",
        "s_rs", "s_ap", "brass_rsp", "brass_rho", "brass_X0", "brass_za", "rs_rsp", "rs_rho", "rs_X0", "rho_min",
        "delta_E")] + [("flags", C.c_int32), ("n_batches", C.c_int32)]


class _Ct(C.Structure):
    _fields_ = [("n", C.c_int32 * 3), ("h", C.c_float * 3), ("origin", C.c_float * 3), ("hu", C.c_void_p),
                ("hu_on_device", C.c_int32)]


class _Calib(C.Structure):
    _fields_ = [("n", C.c_int32), ("hu", C.c_void_p), ("rsp", C.c_void_p), ("rho", C.c_void_p), ("xsp", C.c_void_p)]


class _Frame(C.Structure):
    _fields_ = [("iso", C.c_float * 3), ("rot", C.c_float * 9)]


class Scenario(C.Structure):
    _fields_ = [("shift", C.c_float * 3), ("rsp_scale", C.c_float)]


class _Csr(C.Structure):
    _fields_ = [("row_ptr", C.c_void_p), ("col", C.c_void_p), ("val", C.c_void_p), ("nnz", C.c_int64),
                ("n_rows", C.c_int32)]


class Tallies(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("incident", "dep_ct", "dep_rs", "dep_brass", "escaped", "removed")] + \
               [(n, C.c_uint64) for n in ("n_stopped_ct", "n_stopped_rs", "n_stopped_brass", "n_nuclear", "n_escaped",
                                          "n_steps_ct", "n_steps_dev", "n_steps_slab")]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


class InfluenceStats(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in ("box_elements", "ovf_deposits", "ovf_kept", "columns_replayed", "groups", "nnz")]

    def as_dict(self):
        return {n: int(getattr(self, n)) for n, _ in self._fields_}


STEP_DTYPE = np.dtype([("hid", "<u8"), ("step", "<i4"), ("region", "<i4"), ("cause", "<i4"), ("ivox", "<i4", 3),
                       ("r", "<f4", 3), ("u", "<f4", 3), ("E_before", "<f4"), ("E_after", "<f4"), ("s", "<f4"),
                       ("dep", "<f4"), ("pad_", "<i4")], align=True)

STATE_DTYPE = np.dtype([("hid", "<u8"), ("kind", "<i4"), ("step", "<i4"), ("beam", "<i4"), ("spot", "<i4"),
                        ("ivox", "<i4", 3), ("pad_", "<i4"), ("r", "<f8", 3), ("u", "<f8", 3),
                        ("E", "<f8"), ("t_rad", "<f8"), ("tau", "<f8"), ("tau_star", "<f8")], align=True)
STATE_OUT_DTYPE = np.dtype([("region", "<i4"), ("cause", "<i4"), ("step_after", "<i4"), ("n_steps", "<i4"),
                            ("ivox_after", "<i4", 3), ("pad_", "<i4"), ("r", "<f8", 3), ("u", "<f8", 3),
                            ("E", "<f8"), ("R", "<f8"), ("s", "<f8"), ("dep", "<f8"), ("t_rad", "<f8"), ("tau", "<f8"),
                            ("tau_star", "<f8")], align=True)

DIGEST_DTYPE = np.dtype([("hid", "<u8"), ("hash", "<u8"), ("n_rec", "<i4"), ("cause", "<i4"), ("r", "<f4", 3),
                         ("E_last", "<f4"), ("dep_ct", "<f4"), ("pad_", "<i4")], align=True)

_ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)

_lib = None


def lib():
    """Load libvpmc.so; fails loudly if it has not been built (python -m paper_2307_01416_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libvpmc.so is missing: build it with `python -m paper_2307_01416_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.vpmc_version.restype = C.c_char_p
        L.vpmc_last_error.restype = C.c_char_p
        L.vpmc_last_error.argtypes = [C.c_void_p]
        L.vpmc_default_params.argtypes = [C.POINTER(Params)]
        L.vpmc_default_params.restype = None
        L.vpmc_create.argtypes = [C.POINTER(C.c_void_p), C.POINTER(_Ct), C.POINTER(_Calib), C.POINTER(Params)]
        L.vpmc_destroy.argtypes = [C.c_void_p]
        L.vpmc_add_beam.argtypes = [C.c_void_p, C.POINTER(_Frame), C.POINTER(C.c_int)]
        L.vpmc_set_beam.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_int32]
        L.vpmc_set_range_shifter.argtypes = [C.c_void_p, C.c_int, C.c_float, C.c_float]
        L.vpmc_set_aperture.argtypes = [C.c_void_p, C.c_int, C.c_float, C.c_int, C.c_void_p, C.c_int32, C.c_int32,
                                        C.c_float, C.c_float, C.c_float, C.c_float, C.c_float]
        L.vpmc_dose.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, C.c_void_p, C.c_void_p]
        L.vpmc_dose_scenario.argtypes = [C.c_void_p, C.POINTER(Scenario), C.c_uint64, C.c_uint64, C.c_void_p, C.c_void_p]
        L.vpmc_dose_host.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, C.c_void_p]
        L.vpmc_set_history_window.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64]
        L.vpmc_influence.argtypes = [C.c_void_p, C.POINTER(Scenario), C.c_int32, C.c_uint32, C.c_float, C.c_uint64,
                                     C.POINTER(_Csr), _ALLOC_FN, C.c_void_p, C.c_void_p]
        L.vpmc_csr_from_dense.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_float, C.c_void_p, C.c_void_p,
                                          C.POINTER(C.c_int64)]
        L.vpmc_get_tallies.argtypes = [C.c_void_p, C.POINTER(Tallies)]
        L.vpmc_get_uncertainty.argtypes = [C.c_void_p, C.POINTER(C.c_float)]
        L.vpmc_trace.argtypes = [C.c_void_p, C.POINTER(Scenario), C.c_int32, C.c_uint64, C.c_uint64, C.c_void_p,
                                 C.c_int32, C.c_int32, C.c_void_p, C.c_void_p]
        L.vpmc_get_launch_count.argtypes = [C.c_void_p, C.POINTER(C.c_uint64)]
        L.vpmc_set_timing.argtypes = [C.c_void_p, C.c_int]
        L.vpmc_get_timing.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_uint64)]
        L.vpmc_set_workspace_limit.argtypes = [C.c_void_p, C.c_uint64]
        L.vpmc_step_from_state.argtypes = [C.c_void_p, C.POINTER(Scenario), C.c_uint64, C.c_void_p, C.c_int32, C.c_void_p]
        L.vpmc_set_knob.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.vpmc_dose_to_uncertainty.argtypes = [C.c_void_p, C.POINTER(Scenario), C.c_uint64, C.c_int32, C.c_int32, C.c_float,
                                               C.c_uint64, C.c_void_p, C.c_void_p]
        L.vpmc_get_run_info.argtypes = [C.c_void_p, C.POINTER(C.c_int32), C.POINTER(C.c_float), C.POINTER(C.c_int32)]
        L.vpmc_bench_red.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, C.POINTER(C.c_double), C.POINTER(C.c_uint64)]
        L.vpmc_get_aperture_tables.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.POINTER(C.c_int32)]
        L.vpmc_set_shard.argtypes = [C.c_void_p, C.c_int32, C.c_int32]
        L.vpmc_get_influence_stats.argtypes = [C.c_void_p, C.POINTER(InfluenceStats)]
        L.vpmc_spmv_dose.argtypes = [C.c_void_p, C.POINTER(_Csr), C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p]
        L.vpmc_spmv_grad.argtypes = [C.c_void_p, C.POINTER(_Csr), C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]
        L.vpmc_spmv_grad_static.argtypes = [C.c_void_p, C.POINTER(_Csr), C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]
        L.vpmc_worst_case.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.vpmc_robust_iteration.argtypes = [C.c_void_p, C.POINTER(_Csr), C.c_int32, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                            C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.vpmc_set_aperture_polygon.argtypes = [C.c_void_p, C.c_int, C.c_float, C.c_int, C.c_void_p, C.c_int32, C.c_float]
        L.vpmc_gamma.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_float, C.c_float, C.c_float, C.c_int32, C.POINTER(C.c_uint64),
                                 C.POINTER(C.c_uint64), C.c_void_p]
        L.vpmc_set_scoring_grid.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32]
        L.vpmc_get_scoring_dims.argtypes = [C.c_void_p, C.POINTER(C.c_int32)]
        L.vpmc_digests.argtypes = [C.c_void_p, C.POINTER(Scenario), C.c_uint64, C.c_uint64, C.c_uint64, C.c_int32, C.c_void_p]
        _lib = L
    return _lib


def default_params(**kw) -> Params:
    p = Params()
    lib().vpmc_default_params(C.byref(p))
    for k, v in kw.items():
        if not hasattr(p, k):
            raise KeyError(k)
        setattr(p, k, v)
    return p


def scenario(shift=(0.0, 0.0, 0.0), rsp_scale=1.0) -> Scenario:
    s = Scenario()
    s.shift[:] = [float(x) for x in shift]
    s.rsp_scale = float(rsp_scale)
    return s


def _f32(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float32))


class Engine:
    """One vpmc_t handle.  `problem` is a workload dict (paper_2307_01416_b200.workloads)."""

    def __init__(self, problem: dict, params: Params | None = None):
        self._h = C.c_void_p()
        L = lib()
        ct = problem["ct"]
        hu = np.ascontiguousarray(np.asarray(ct["hu"], dtype=np.int16).reshape(-1))
        c = _Ct()
        c.n[:] = [int(x) for x in ct["n"]]
        c.h[:] = [float(x) for x in ct["h"]]
        c.origin[:] = [float(x) for x in ct["origin"]]
        c.hu = hu.ctypes.data
        c.hu_on_device = 0
        cal = problem["calib"]
        arrs = {k: (None if cal.get(k) is None else _f32(cal[k])) for k in ("hu", "rsp", "rho", "xsp")}
        k = _Calib()
        k.n = int(arrs["hu"].size)
        k.hu, k.rsp, k.rho = arrs["hu"].ctypes.data, arrs["rsp"].ctypes.data, arrs["rho"].ctypes.data
        k.xsp = None if arrs["xsp"] is None else arrs["xsp"].ctypes.data
        rc = L.vpmc_create(C.byref(self._h), C.byref(c), C.byref(k), C.byref(params) if params is not None else None)
        if rc != OK:
            raise VpmcError(rc, L.vpmc_last_error(None).decode())
        self.n = tuple(int(x) for x in ct["n"])
        self.nvox = self.n[0] * self.n[1] * self.n[2]
        self.ncell = self.nvox              # elements of a dose grid (vpmc_set_scoring_grid changes it)
        self.h2d_bytes = hu.nbytes + sum(a.nbytes for a in arrs.values() if a is not None)
        self.n_spots = 0
        for b in problem["beams"]:
            self.add_beam(b)

    # -- plumbing
    def _check(self, rc):
        if rc != OK:
            raise VpmcError(rc, lib().vpmc_last_error(self._h).decode())

    def close(self):
        if self._h:
            lib().vpmc_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- set-up (S0)
    def add_beam(self, b: dict) -> int:
        L = lib()
        f = _Frame()
        f.iso[:] = [float(x) for x in b["iso"]]
        f.rot[:] = [float(x) for x in np.asarray(b["rot"], dtype=np.float32).reshape(9)]
        bid = C.c_int(-1)
        self._check(L.vpmc_add_beam(self._h, C.byref(f), C.byref(bid)))
        sp = _f32(b["spots"]).reshape(-1, 5)
        self._check(L.vpmc_set_beam(self._h, bid.value, sp.ctypes.data, sp.shape[0]))
        self.n_spots += sp.shape[0]
        self.h2d_bytes += sp.nbytes
        if float(b.get("rs_wet", 0.0)) > 0:
            self._check(L.vpmc_set_range_shifter(self._h, bid.value, float(b["rs_wet"]), float(b.get("rs_face", 190.0))))
        ap = b.get("aperture")
        if ap is not None and ap.get("polygon") is not None:
            poly = _f32(ap["polygon"]).reshape(-1, 2)
            self._check(L.vpmc_set_aperture_polygon(self._h, bid.value, float(ap["T"]), BRASS, poly.ctypes.data, poly.shape[0],
                                                    float(ap.get("face", 150.0))))
            self.h2d_bytes += poly.nbytes
        elif ap is not None:
            op = np.ascontiguousarray(np.asarray(ap["open"], dtype=np.uint8))
            self._check(L.vpmc_set_aperture(self._h, bid.value, float(ap["T"]), BRASS, op.ctypes.data, op.shape[1],
                                            op.shape[0], float(ap["u0"]), float(ap["v0"]), float(ap["du"]),
                                            float(ap["dv"]), float(ap.get("face", 150.0))))
            self.h2d_bytes += op.nbytes
        return bid.value

    def set_history_window(self, begin: int, end: int):
        self._check(lib().vpmc_set_history_window(self._h, int(begin), int(end)))

    def set_scoring_grid(self, div=(1, 1, 1)):
        """Score on cells of div voxels per axis (vpmc_set_scoring_grid); returns the scoring grid's dimensions."""
        self._check(lib().vpmc_set_scoring_grid(self._h, int(div[0]), int(div[1]), int(div[2])))
        d = (C.c_int32 * 3)()
        self._check(lib().vpmc_get_scoring_dims(self._h, d))
        self.ncell = int(d[0]) * int(d[1]) * int(d[2])
        return int(d[0]), int(d[1]), int(d[2])

    def set_shard(self, index: int, count: int):
        """This handle computes shard `index` of `count` (vpmc_set_shard)."""
        self._check(lib().vpmc_set_shard(self._h, int(index), int(count)))

    # -- hot path
    def dose(self, n_histories: int, seed: int, out=None, sc: Scenario | None = None, stream=None):
        """Dose [Gy] as a torch.float32 CUDA tensor of nvox elements (v = ix + nx*(iy + ny*iz))."""
        import torch
        if out is None:
            out = torch.empty(self.ncell, dtype=torch.float32, device="cuda")
        assert out.is_cuda and out.dtype == torch.float32 and out.numel() == self.ncell and out.is_contiguous()
        st = torch.cuda.current_stream() if stream is None else stream
        if sc is None:
            self._check(lib().vpmc_dose(self._h, int(n_histories), int(seed), out.data_ptr(), st.cuda_stream))
        else:
            self._check(lib().vpmc_dose_scenario(self._h, C.byref(sc), int(n_histories), int(seed), out.data_ptr(),
                                                 st.cuda_stream))
        return out

    def dose_to_uncertainty(self, batch_histories: int, target: float, seed: int, min_batches: int = 2,
                            max_batches: int = 1000, out=None, sc: Scenario | None = None, stream=None):
        """Dose run batch by batch until the C6 estimate <= target, the stopping rule decided on the device
        (vpmc_dose_to_uncertainty).  Returns the dose tensor; run_info() gives (batches, estimate, reached)."""
        import torch
        if out is None:
            out = torch.empty(self.ncell, dtype=torch.float32, device="cuda")
        assert out.is_cuda and out.dtype == torch.float32 and out.numel() == self.ncell and out.is_contiguous()
        st = torch.cuda.current_stream() if stream is None else stream
        self._check(lib().vpmc_dose_to_uncertainty(self._h, C.byref(sc) if sc is not None else None, int(batch_histories),
                                                   int(min_batches), int(max_batches), float(target), int(seed),
                                                   out.data_ptr(), st.cuda_stream))
        return out

    def run_info(self):
        b, u, r = C.c_int32(), C.c_float(), C.c_int32()
        self._check(lib().vpmc_get_run_info(self._h, C.byref(b), C.byref(u), C.byref(r)))
        return int(b.value), float(u.value), bool(r.value)

    def dose_host(self, n_histories: int, seed: int, out: np.ndarray | None = None) -> np.ndarray:
        if out is None:
            out = np.empty(self.ncell, dtype=np.float32)
        assert out.size == self.ncell
        self._check(lib().vpmc_dose_host(self._h, int(n_histories), int(seed), out.ctypes.data))
        return out

    def tallies(self) -> Tallies:
        t = Tallies()
        self._check(lib().vpmc_get_tallies(self._h, C.byref(t)))
        return t

    def uncertainty(self) -> float:
        u = C.c_float()
        self._check(lib().vpmc_get_uncertainty(self._h, C.byref(u)))
        return float(u.value)

    def launch_count(self) -> int:
        n = C.c_uint64()
        self._check(lib().vpmc_get_launch_count(self._h, C.byref(n)))
        return int(n.value)

    def set_timing(self, on: bool):
        self._check(lib().vpmc_set_timing(self._h, 1 if on else 0))

    def timing(self):
        """{class: (milliseconds, launches)} accumulated since the last call; classes beamline (persistent beam kernels) /
        voxel / scoring / writer / stage (one-thread-per-item source, aperture-entry and CT-entry kernels)."""
        ms = (C.c_double * 6)()
        n = (C.c_uint64 * 6)()
        self._check(lib().vpmc_get_timing(self._h, ms, n))
        return {k: (float(ms[i]), int(n[i])) for i, k in enumerate(("beamline", "voxel", "scoring", "writer", "stage", "optimiser"))}

    def trace(self, hids, n_or_hps: int, seed: int, sc: Scenario | None = None, mode: int = 0, max_steps: int = 1024):
        hids = np.ascontiguousarray(np.asarray(hids, dtype=np.uint64))
        recs = np.zeros((hids.size, max_steps), dtype=STEP_DTYPE)
        nrec = np.zeros(hids.size, dtype=np.int32)
        self._check(lib().vpmc_trace(self._h, C.byref(sc) if sc is not None else None, mode, int(n_or_hps), int(seed),
                                     hids.ctypes.data, hids.size, max_steps, recs.ctypes.data, nrec.ctypes.data))
        assert (nrec <= max_steps).all(), "max_steps too small"
        return [recs[i, :nrec[i]] for i in range(hids.size)]

    def influence(self, scenarios, hist_per_spot: int, rel_threshold: float, seed: int, stream=None):
        """List of (row_ptr int64, col int32, val fp32) torch CUDA tensors, one per scenario."""
        import torch
        st = torch.cuda.current_stream() if stream is None else stream
        keep = {}

        def _alloc(nbytes, _user):
            t = torch.empty(max(int(nbytes), 1), dtype=torch.uint8, device="cuda")
            keep[t.data_ptr()] = t
            return t.data_ptr()

        cb = _ALLOC_FN(_alloc)
        n_sc = len(scenarios)
        arr = (Scenario * n_sc)(*scenarios)
        out = (_Csr * n_sc)()
        self._check(lib().vpmc_influence(self._h, arr, n_sc, int(hist_per_spot), float(rel_threshold), int(seed), out, cb,
                                         None, st.cuda_stream))
        res = []
        for o in out:
            rp = keep[o.row_ptr][: 8 * (o.n_rows + 1)].view(torch.int64)
            col = keep[o.col][: 4 * o.nnz].view(torch.int32) if o.nnz else torch.empty(0, dtype=torch.int32, device="cuda")
            val = keep[o.val][: 4 * o.nnz].view(torch.float32) if o.nnz else torch.empty(0, dtype=torch.float32, device="cuda")
            res.append((rp, col, val))
        return res

    # -- optimiser iteration on the CSR matrices (marshalling only; the products run in vpmc_spmv.cuh)
    @staticmethod
    def _csr(m) -> _Csr:
        import torch
        rp, col, val = m
        assert rp.is_cuda and rp.dtype == torch.int64 and col.dtype == torch.int32 and val.dtype == torch.float32
        assert rp.is_contiguous() and col.is_contiguous() and val.is_contiguous()
        c = _Csr()
        c.row_ptr, c.col, c.val = rp.data_ptr(), col.data_ptr() if col.numel() else None, val.data_ptr() if val.numel() else None
        c.nnz, c.n_rows = int(col.numel()), int(rp.numel()) - 1
        return c

    def spmv_dose(self, m, w, n_cols: int | None = None, out=None, stream=None):
        """dose[v] = sum_j D[j][v] w[j] for a CSR matrix m = (row_ptr, col, val) of CUDA tensors (rows = spots)."""
        import torch
        n_cols = self.ncell if n_cols is None else int(n_cols)
        if out is None:
            out = torch.empty(n_cols, dtype=torch.float32, device="cuda")
        assert w.is_cuda and w.dtype == torch.float32 and w.is_contiguous() and out.numel() == n_cols
        st = torch.cuda.current_stream() if stream is None else stream
        c = self._csr(m)
        self._check(lib().vpmc_spmv_dose(self._h, C.byref(c), n_cols, w.data_ptr(), out.data_ptr(), st.cuda_stream))
        return out

    def spmv_grad(self, m, r, out=None, accumulate: bool = False, stream=None):
        """grad[j] (+)= sum_v D[j][v] r[v]."""
        import torch
        c = self._csr(m)
        if out is None:
            assert not accumulate
            out = torch.empty(c.n_rows, dtype=torch.float32, device="cuda")
        assert r.is_cuda and r.dtype == torch.float32 and r.is_contiguous() and out.numel() == c.n_rows
        st = torch.cuda.current_stream() if stream is None else stream
        self._check(lib().vpmc_spmv_grad(self._h, C.byref(c), r.data_ptr(), out.data_ptr(), 1 if accumulate else 0, st.cuda_stream))
        return out

    def spmv_grad_static(self, m, r, out, accumulate: bool = False, stream=None):
        """vpmc_spmv_grad_static: spmv_grad with the library's static scratch -- no device allocation inside the call, so `out`
        (n_rows floats) is the caller's; at most STATIC_MAX_NNZ entries; calls that overlap on the GPU race on the scratch."""
        import torch
        c = self._csr(m)
        assert r.is_cuda and r.dtype == torch.float32 and r.is_contiguous()
        assert out.is_cuda and out.dtype == torch.float32 and out.is_contiguous() and out.numel() == c.n_rows
        st = torch.cuda.current_stream() if stream is None else stream
        self._check(lib().vpmc_spmv_grad_static(self._h, C.byref(c), r.data_ptr(), out.data_ptr(), 1 if accumulate else 0, st.cuda_stream))
        return out

    def worst_case(self, doses, target, weight, stream=None):
        """(objective 0-d float64 CUDA tensor, resid [n_sc, n]) of the voxel-wise worst case over the rows of doses [n_sc, n]."""
        import torch
        assert doses.is_cuda and doses.dtype == torch.float32 and doses.is_contiguous() and doses.dim() == 2
        n_sc, n = doses.shape
        assert target.numel() == n and weight.numel() == n and target.dtype == torch.float32 and weight.dtype == torch.float32
        resid = torch.empty_like(doses)
        obj = torch.zeros((), dtype=torch.float64, device="cuda")
        st = torch.cuda.current_stream() if stream is None else stream
        self._check(lib().vpmc_worst_case(self._h, doses.data_ptr(), n_sc, n, target.data_ptr(), weight.data_ptr(), resid.data_ptr(),
                                          obj.data_ptr(), st.cuda_stream))
        return obj, resid

    def robust_iteration(self, mats, w, target, weight, ws=None, stream=None):
        """One optimiser iteration on the scenario matrices `mats`: (objective 0-d float64 tensor, grad [n_spots], doses [n_sc, nvox]).
        ws = (doses, resid) workspaces from an earlier call, reused."""
        import torch
        n_sc, n = len(mats), int(target.numel())
        arr = (_Csr * n_sc)(*[self._csr(m) for m in mats])
        if ws is None:
            ws = (torch.empty((n_sc, n), dtype=torch.float32, device="cuda"), torch.empty((n_sc, n), dtype=torch.float32, device="cuda"))
        doses, resid = ws
        grad = torch.empty(arr[0].n_rows, dtype=torch.float32, device="cuda")
        obj = torch.zeros((), dtype=torch.float64, device="cuda")
        assert w.is_cuda and w.dtype == torch.float32 and w.numel() == arr[0].n_rows
        st = torch.cuda.current_stream() if stream is None else stream
        self._check(lib().vpmc_robust_iteration(self._h, arr, n_sc, n, w.data_ptr(), target.data_ptr(), weight.data_ptr(), doses.data_ptr(),
                                                resid.data_ptr(), grad.data_ptr(), obj.data_ptr(), st.cuda_stream))
        return obj, grad, doses

    def gamma(self, ref, ev, dd: float = 0.01, dta: float = 1.0, thr: float = 0.1, sub: int = 10, stream=None):
        """3-D gamma of two dose tensors on this engine's grid (vpmc_gamma): (pass rate, voxels evaluated, voxels failing)."""
        import torch
        for t in (ref, ev):
            assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and t.numel() == self.ncell
        st = torch.cuda.current_stream() if stream is None else stream
        ne, nf = C.c_uint64(), C.c_uint64()
        self._check(lib().vpmc_gamma(self._h, ref.data_ptr(), ev.data_ptr(), float(dd), float(dta), float(thr), int(sub), C.byref(ne),
                                     C.byref(nf), st.cuda_stream))
        return (1.0 - nf.value / ne.value) if ne.value else 1.0, int(ne.value), int(nf.value)

    def influence_stats(self) -> dict:
        st = InfluenceStats()
        self._check(lib().vpmc_get_influence_stats(self._h, C.byref(st)))
        return st.as_dict()

    def step_from_state(self, states: np.ndarray, seed: int, sc: Scenario | None = None) -> np.ndarray:
        """Test-only: one step from each pre-step state (STATE_DTYPE array) -> STATE_OUT_DTYPE array."""
        states = np.ascontiguousarray(states, dtype=STATE_DTYPE)
        out = np.zeros(states.size, dtype=STATE_OUT_DTYPE)
        self._check(lib().vpmc_step_from_state(self._h, C.byref(sc) if sc is not None else None, int(seed),
                                               states.ctypes.data, states.size, out.ctypes.data))
        return out

    def digests(self, n_histories: int, seed: int, hid_begin: int, n: int, sc: Scenario | None = None) -> np.ndarray:
        """Test-only: DIGEST_DTYPE array of the history ids [hid_begin, hid_begin + n) of the n_histories-history run."""
        out = np.zeros(n, dtype=DIGEST_DTYPE)
        self._check(lib().vpmc_digests(self._h, C.byref(sc) if sc is not None else None, int(n_histories), int(seed),
                                       int(hid_begin), int(n), out.ctypes.data))
        return out

    def aperture_tables(self, beam: int = 0):
        """Test-only: (packed bitmap uint32 [rows, words], distance maps uint8 [2, tiles_v, tiles_u]) of a beam's aperture."""
        dims = (C.c_int32 * 4)()
        self._check(lib().vpmc_get_aperture_tables(self._h, int(beam), None, None, dims))
        bits = np.zeros((dims[1], dims[0]), dtype=np.uint32)
        dist = np.zeros((2, dims[3], dims[2]), dtype=np.uint8)
        self._check(lib().vpmc_get_aperture_tables(self._h, int(beam), bits.ctypes.data, dist.ctypes.data, dims))
        return bits, dist

    def bench_red(self, buffer_bytes: int = 4 << 20, n_ops: int = 1 << 30):
        """fp32 REDs per second into an L2-resident buffer of buffer_bytes (vpmc_bench_red): (ops/s, ops issued)."""
        ms, n = C.c_double(), C.c_uint64()
        self._check(lib().vpmc_bench_red(self._h, int(buffer_bytes), int(n_ops), C.byref(ms), C.byref(n)))
        return n.value / (ms.value * 1e-3), int(n.value)

    def set_knob(self, knob: int, value: float):
        self._check(lib().vpmc_set_knob(self._h, int(knob), float(value)))

    def set_workspace_limit(self, nbytes: int):
        self._check(lib().vpmc_set_workspace_limit(self._h, int(nbytes)))

    def csr_from_dense(self, col, rel_threshold: float):
        """The CSR writer alone on one dense fp32 CUDA column: (idx int32, val fp32) CUDA tensors."""
        import torch
        assert col.is_cuda and col.dtype == torch.float32 and col.is_contiguous()
        nnz = C.c_int64()
        self._check(lib().vpmc_csr_from_dense(self._h, col.data_ptr(), col.numel(), float(rel_threshold), None, None,
                                              C.byref(nnz)))
        idx = torch.empty(max(nnz.value, 1), dtype=torch.int32, device=col.device)
        val = torch.empty(max(nnz.value, 1), dtype=torch.float32, device=col.device)
        n2 = C.c_int64()
        self._check(lib().vpmc_csr_from_dense(self._h, col.data_ptr(), col.numel(), float(rel_threshold), idx.data_ptr(),
                                              val.data_ptr(), C.byref(n2)))
        assert n2.value == nnz.value
        return idx[: nnz.value], val[: nnz.value]
