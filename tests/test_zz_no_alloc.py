"""vpmc_spmv_grad_static (include/vpmc.h): the entry point that allocates nothing -- the gradient gather of the optimiser
iteration with its scratch in a file-scope device array of the library -- against the existing path vpmc_spmv_grad (scratch
from the buffer cache) and the oracle.  Two calls in a row on different matrices: the array keeps the first call's contents and
the second result must not depend on them.  Same kernels, same order: the results are bit-equal; the bar asserted first is the
one tests/test_gpu_spmv.py uses (1e-6 of the sum of the absolute terms).
This file sorts last on purpose (the suite runs with pytest -x); it must pass alone in a fresh process and after the others."""
import ctypes as C

import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

CH = 8192            # kSpmvChunk


def _csr(rng, lengths, n_cols):
    rp = np.concatenate([[0], np.cumsum(lengths)]).astype(np.int64)
    col = np.empty(rp[-1], dtype=np.int32)
    for j, n in enumerate(lengths):
        if n:
            start = int(rng.integers(0, n_cols - 2 * n))
            col[rp[j]:rp[j + 1]] = np.sort(rng.choice(np.arange(start, start + 2 * n), size=n, replace=False))
    val = (rng.random(rp[-1]) * 2.0 + 0.01).astype(np.float32)
    return rp, col, val


def _engine():
    from paper_2307_01416_b200 import binding, workloads as wl
    return binding, binding.Engine(wl.small_water(n=(8, 8, 20)))


def test_static_scratch_gradient_equals_the_existing_path_twice_in_a_row():
    from oracle import robust_oracle as rob
    binding, eng = _engine()
    rng = np.random.default_rng(41)
    n_cols = 300_007
    # rows across several chunks, empty rows, rows on chunk borders, a ragged tail; the second matrix is cut differently
    cases = ([3 * CH + 17, 5, 0, 0, 2 * CH - 5, 1, CH, 40000, 0, 77], [CH, CH, 13, 0, 5 * CH + 1, 900, 2 * CH])
    mats = [_csr(rng, ln, n_cols) for ln in cases]
    dev = [tuple(torch.from_numpy(a).cuda() for a in m) for m in mats]
    rs = [torch.from_numpy(rng.standard_normal(n_cols).astype(np.float32)).cuda() for _ in mats]
    ref = [eng.spmv_grad(m, r).clone() for m, r in zip(dev, rs)]                  # the existing path
    outs = [torch.full((len(ln),), 7.0, dtype=torch.float32, device="cuda") for ln in cases]
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for m, r, o in zip(dev, rs, outs):                                            # two calls in a row, nothing in between
        eng.spmv_grad_static(m, r, o)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0                                  # no device memory was taken
    for m, r, o, g in zip(mats, rs, outs, ref):
        g_abs = rob.spmv_grad((m[0], m[1], np.abs(m[2])), np.abs(r.cpu().numpy()))
        assert np.all(np.abs(o.cpu().numpy().astype(np.float64) - g.cpu().numpy().astype(np.float64)) <= 1e-6 * g_abs + 1e-30)
        assert torch.equal(o, g)                                                  # same kernels, same order
        assert np.all(np.abs(o.cpu().numpy().astype(np.float64) - rob.spmv_grad(m, r.cpu().numpy())) <= 1e-6 * g_abs + 1e-30)
    # accumulate, and the first matrix again after the second (stale partial sums of a longer matrix in the array)
    acc = torch.full_like(outs[0], 3.0)
    eng.spmv_grad_static(dev[0], rs[0], acc, accumulate=True)
    want = eng.spmv_grad(dev[0], rs[0], out=torch.full_like(outs[0], 3.0), accumulate=True)
    assert torch.equal(acc, want)
    eng.close()


def test_static_scratch_rejects_what_it_cannot_hold_and_serves_empty_inputs():
    binding, eng = _engine()
    L = binding.lib()
    rp = torch.zeros(2, dtype=torch.int64, device="cuda")
    one = torch.zeros(1, dtype=torch.float32, device="cuda")
    idx = torch.zeros(1, dtype=torch.int32, device="cuda")
    big = binding._Csr()
    big.row_ptr, big.col, big.val, big.nnz, big.n_rows = rp.data_ptr(), idx.data_ptr(), one.data_ptr(), binding.STATIC_MAX_NNZ + 1, 1
    assert L.vpmc_spmv_grad_static(eng._h, C.byref(big), one.data_ptr(), one.data_ptr(), 0, None) == binding.ERR_INVALID_ARG
    msg = L.vpmc_last_error(eng._h)
    msg = msg.decode() if isinstance(msg, bytes) else str(msg)
    assert "VPMC_STATIC_MAX_NNZ" in msg
    assert L.vpmc_spmv_grad_static(eng._h, None, one.data_ptr(), one.data_ptr(), 0, None) == binding.ERR_INVALID_ARG
    # a matrix without entries: the rows are set to zero (or left alone when accumulating), as in vpmc_spmv_grad
    empty = (torch.zeros(4, dtype=torch.int64, device="cuda"), torch.zeros(0, dtype=torch.int32, device="cuda"),
             torch.zeros(0, dtype=torch.float32, device="cuda"))
    out = torch.full((3,), 5.0, dtype=torch.float32, device="cuda")
    eng.spmv_grad_static(empty, one, out)
    assert torch.equal(out, torch.zeros_like(out))
    out.fill_(5.0)
    eng.spmv_grad_static(empty, one, out, accumulate=True)
    assert torch.equal(out, torch.full_like(out, 5.0))
    # the handle still works afterwards
    assert float(eng.dose(2000, 1).sum()) > 0
    eng.close()
