"""Error behaviour of the C-ABI as include/vpmc.h states it: every call returns VPMC_OK or a negative VPMC_ERR_*, nothing
throws or aborts, vpmc_last_error gives a message, and a handle stays usable after a rejected call."""
import ctypes as C

import numpy as np
import pytest
import torch

from paper_2307_01416_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _eng():
    from paper_2307_01416_b200 import binding
    return binding, binding.Engine(wl.small_water(n=(8, 8, 20), with_aperture=True))


def test_rejected_calls_report_and_leave_the_handle_usable():
    b, eng = _eng()
    L = b.lib()
    h = eng._h
    d = torch.zeros(eng.nvox, dtype=torch.float32, device="cuda")
    one = torch.ones(4, dtype=torch.float32, device="cuda")
    ne, nf = C.c_uint64(), C.c_uint64()
    bad = [
        L.vpmc_set_scoring_grid(h, 0, 1, 1), L.vpmc_set_scoring_grid(h, 1, 9, 1),                      # divisors outside [1, n]
        L.vpmc_set_shard(h, 2, 2), L.vpmc_set_shard(h, 0, 0), L.vpmc_set_shard(h, -1, 3),
        L.vpmc_gamma(h, d.data_ptr(), d.data_ptr(), C.c_float(0.0), C.c_float(1.0), C.c_float(0.1), 10, C.byref(ne), C.byref(nf), None),
        L.vpmc_gamma(h, d.data_ptr(), None, C.c_float(0.01), C.c_float(1.0), C.c_float(0.1), 10, C.byref(ne), C.byref(nf), None),
        L.vpmc_gamma(h, d.data_ptr(), d.data_ptr(), C.c_float(0.01), C.c_float(1.0), C.c_float(0.1), 0, C.byref(ne), C.byref(nf), None),
        L.vpmc_spmv_dose(h, None, eng.nvox, one.data_ptr(), d.data_ptr(), None),
        L.vpmc_worst_case(h, d.data_ptr(), 0, eng.nvox, d.data_ptr(), d.data_ptr(), d.data_ptr(), d.data_ptr(), None),
        L.vpmc_set_knob(h, 99, 1.0), L.vpmc_set_knob(h, b.KNOB_CHUNK, 3.0),
        L.vpmc_dose(h, 1000, 1, None, None),
        L.vpmc_dose_to_uncertainty(h, None, 0, 2, 10, C.c_float(0.01), 1, d.data_ptr(), None),
        L.vpmc_bench_red(h, 3000, 1000, None, None),
    ]
    assert all(rc == b.ERR_INVALID_ARG for rc in bad), bad
    assert len(L.vpmc_last_error(h).decode()) > 0
    # a CSR whose scenarios disagree in their row counts
    rp3 = torch.zeros(4, dtype=torch.int64, device="cuda"); rp2 = torch.zeros(3, dtype=torch.int64, device="cuda")
    e = torch.zeros(0, dtype=torch.int32, device="cuda"); ev = torch.zeros(0, dtype=torch.float32, device="cuda")
    w = torch.ones(3, dtype=torch.float32, device="cuda")
    with pytest.raises(b.VpmcError) as ei:
        eng.robust_iteration([(rp3, e, ev), (rp2, e, ev)], w, d, d)
    assert ei.value.code == b.ERR_INVALID_ARG and "rows" in str(ei.value)
    # state errors: results asked for before the run that produces them
    with pytest.raises(b.VpmcError) as ei:
        eng.run_info()
    assert ei.value.code == b.ERR_STATE
    with pytest.raises(b.VpmcError) as ei:
        eng.uncertainty()
    assert ei.value.code == b.ERR_STATE
    # the handle still works
    out = eng.dose(5000, 1)
    assert bool(torch.isfinite(out).all()) and float(out.sum()) > 0 and eng.uncertainty() > 0
    assert L.vpmc_destroy(None) == b.OK and L.vpmc_set_shard(None, 0, 1) == b.ERR_INVALID_ARG
    eng.close()


def test_empty_optimiser_inputs():
    """Matrices without entries, rows without entries: products are zeros, the objective is the target's own deviation."""
    b, eng = _eng()
    n = eng.nvox
    rp = torch.zeros(6, dtype=torch.int64, device="cuda")
    m = (rp, torch.zeros(0, dtype=torch.int32, device="cuda"), torch.zeros(0, dtype=torch.float32, device="cuda"))
    w = torch.ones(5, dtype=torch.float32, device="cuda")
    t = torch.full((n,), 2.0, dtype=torch.float32, device="cuda"); p = torch.ones(n, dtype=torch.float32, device="cuda")
    assert float(eng.spmv_dose(m, w).abs().max()) == 0.0
    assert float(eng.spmv_grad(m, t).abs().max()) == 0.0
    obj, grad, doses = eng.robust_iteration([m, m], w, t, p)
    assert abs(float(obj) - 4.0 * n) < 1e-6 * n and float(grad.abs().max()) == 0.0 and float(doses.abs().max()) == 0.0
    eng.close()
