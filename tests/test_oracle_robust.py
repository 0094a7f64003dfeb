"""Pins of the robust-optimiser oracle (oracle/robust_oracle.c, R16) against what the mathematics
fixes: dense numpy products (a library routine on the densified matrix), the adjoint identity, a finite difference of the
objective, and hand-computed cases.  A transposed operand, a dropped factor 2, a wrong sign or a wrong worst-scenario rule
fails one of them."""
import numpy as np

from oracle import robust_oracle as rob


def _random_csr(rng, n_rows, n_cols, density):
    dense = (rng.random((n_rows, n_cols)) < density) * rng.random((n_rows, n_cols))
    dense = dense.astype(np.float32)
    rp = np.zeros(n_rows + 1, dtype=np.int64)
    cols, vals = [], []
    for j in range(n_rows):
        idx = np.nonzero(dense[j])[0]
        cols.append(idx.astype(np.int32)); vals.append(dense[j, idx])
        rp[j + 1] = rp[j] + idx.size
    return (rp, np.concatenate(cols), np.concatenate(vals)), dense.astype(np.float64)


def test_spmv_against_dense_products():
    rng = np.random.default_rng(1)
    for (nr, nc, dens) in ((1, 1, 1.0), (7, 50, 0.3), (40, 333, 0.05), (5, 64, 0.0)):
        m, D = _random_csr(rng, nr, nc, dens)
        w = rng.random(nr); r = rng.standard_normal(nc)
        assert np.allclose(rob.spmv_dose(m, nc, w), D.T @ w, rtol=1e-13, atol=1e-15)      # rows are spots: dose = D^T-layout scatter
        assert np.allclose(rob.spmv_grad(m, r), D @ r, rtol=1e-13, atol=1e-15)
        g0 = rng.random(nr)
        assert np.allclose(rob.spmv_grad(m, r, g0.copy()), g0 + D @ r, rtol=1e-13, atol=1e-15)
    # an asymmetric hand case: row 0 = {v1: 2}, row 1 = {v0: 3, v2: 5}
    m = (np.array([0, 1, 3]), np.array([1, 0, 2], dtype=np.int32), np.array([2, 3, 5], dtype=np.float32))
    assert list(rob.spmv_dose(m, 3, [10.0, 1.0])) == [3.0, 20.0, 5.0]
    assert list(rob.spmv_grad(m, [1.0, 10.0, 100.0])) == [20.0, 503.0]


def test_adjoint_identity():
    rng = np.random.default_rng(2)
    m, _ = _random_csr(rng, 23, 211, 0.1)
    w = rng.random(23); r = rng.standard_normal(211)
    assert abs(rob.spmv_dose(m, 211, w) @ r - w @ rob.spmv_grad(m, r)) < 1e-12 * abs(w @ rob.spmv_grad(m, r))


def test_worst_case_by_hand():
    # 2 scenarios, 3 voxels, target 1, weights (1, 2, 0)
    doses = np.array([[1.5, 0.0, 9.0], [0.0, 1.0, 1.0]])
    f, resid, worst = rob.worst_case(doses, np.ones(3), np.array([1.0, 2.0, 0.0]))
    # voxel 0: e = (+0.5, -1.0) -> scenario 1; voxel 1: e = (-1, 0) -> scenario 0; voxel 2: weight 0
    assert list(worst) == [1, 0, 0]
    assert f == 1.0 * 1.0 + 2.0 * 1.0
    assert np.array_equal(resid, np.array([[0.0, -4.0, 0.0], [-2.0, 0.0, 0.0]]))
    # equal squared deviations: the lowest scenario index is taken
    f, resid, worst = rob.worst_case(np.array([[2.0], [0.0], [2.0]]), np.ones(1), np.ones(1))
    assert list(worst) == [0] and f == 1.0 and resid[0, 0] == 2.0 and resid[1, 0] == 0.0 and resid[2, 0] == 0.0


def test_gradient_is_the_derivative_of_the_objective():
    rng = np.random.default_rng(3)
    nr, nc, ns = 9, 120, 4
    mats = [_random_csr(rng, nr, nc, 0.3)[0] for _ in range(ns)]
    w = rng.random(nr) + 0.5
    t = rng.random(nc) * 3.0; p = rng.random(nc)
    f, g, doses = rob.iteration(mats, nc, w, t, p)
    assert f > 0 and doses.shape == (ns, nc)
    h = 1e-6
    for j in range(nr):
        wp, wm = w.copy(), w.copy()
        wp[j] += h; wm[j] -= h
        fd = (rob.iteration(mats, nc, wp, t, p)[0] - rob.iteration(mats, nc, wm, t, p)[0]) / (2 * h)
        assert abs(fd - g[j]) <= 1e-5 * max(abs(g[j]), 1.0), (j, fd, g[j])      # s* is locally constant away from ties
    # one scenario: plain weighted least squares, closed form 2 D diag(p) (D^T w - t)
    D = np.zeros((nr, nc)); rp, col, val = mats[0]
    for j in range(nr):
        D[j, col[rp[j]:rp[j + 1]]] = val[rp[j]:rp[j + 1]]
    f1, g1, _ = rob.iteration(mats[:1], nc, w, t, p)
    assert np.allclose(g1, 2.0 * D @ (p * (D.T @ w - t)), rtol=1e-12)
    assert abs(f1 - float(p @ (D.T @ w - t) ** 2)) < 1e-12 * f1
