"""GPU parity of the influence path (S7, S8): per-spot columns under scenarios and the CSR writer.

Tolerances:
  * (i) the writer alone is bit-exact: fed the oracle's fp32 column it returns the oracle's (col, val) row;
  * (ii) end to end, the kept sets are equal except for entries whose value lies within +-0.1 % of the threshold
    (counted) -- and except in voxels visited by a RE-DEALT history: a history whose discrete trace differs between
    the two paths (a near-tie flip, tests/test_gpu_parity.py) moves its own deposits.  Those histories are found by
    tracing every history of the column on both sides, counted and bounded, and the voxels either version of them
    visits are the only ones exempt; everywhere else values agree to 1e-5 of the column maximum (fp32 sums);
  * row order, index order, uniqueness and types are always exact; the 1e-3 dose bar holds on the weighted sum of the
    columns (= the plan dose of all H n_spots histories).
"""
import numpy as np
import pytest

from paper_2307_01416_b200 import workloads as wl
from tests.helpers import oracle_problem
from tests.test_gpu_parity import hetero_case, rs_case, rotated_case

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def bind():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2307_01416_b200 import binding
    binding.lib()
    return binding


def orc():
    from oracle import vpmc_oracle
    return vpmc_oracle


def check_csr_structure(rp, col, val, n_rows, nvox):
    assert rp.dtype == np.int64 and col.dtype == np.int32 and val.dtype == np.float32
    assert rp.shape == (n_rows + 1,) and rp[0] == 0 and (np.diff(rp) >= 0).all() and rp[-1] == col.size == val.size
    for r in range(n_rows):
        c = col[rp[r]:rp[r + 1]]
        assert (np.diff(c) > 0).all()                      # ascending voxel index, unique
        assert c.size == 0 or (c[0] >= 0 and c[-1] < nvox)
    assert (val > 0).all()


DRIFT_MM = 1e-5       # a history is "drifted" once its traced position differs from the oracle's by more than this (0.01 um)
S_MAX = 15.0          # MeV / mm of water: stopping power at the R_cut energy (2.35 MeV), the largest a step can see


def flagged_histories(bind, eng, O, pb, g, hps, seed, sc, nvox, n_xy, chunk=2500):
    """Traces every history of column g on both sides.  A history is FLAGGED when its discrete trace differs (a near-tie
    flip, after which its random deflections are re-dealt) or when its position has drifted by more than DRIFT_MM (the
    accumulated difference of DESIGN.md 4.2); every other history is the oracle's history up to the energy a 0.01 um
    shift of a voxel boundary moves (DRIFT_MM x stopping power).  Returns (#re-dealt, #drifted, E_dep difference CUDA - oracle of the flagged histories per voxel [MeV],
    mask of the voxels they visit)."""
    delta = np.zeros(nvox, dtype=np.float64)
    mask = np.zeros(nvox, dtype=bool)
    n_re = n_drift = 0
    sc_g = bind.scenario(sc[0], sc[1])
    sc_o = O.scenario(sc[0], float(np.float32(sc[1])))
    gamma_loc = float(pb.params.gamma_loc)
    for i0 in range(0, hps, chunk):
        hids = np.uint64(g) * np.uint64(hps) + np.arange(i0, min(i0 + chunk, hps), dtype=np.uint64)
        a_all = eng.trace(hids, hps, seed, sc=sc_g, mode=1, max_steps=1000)
        b_all = O.trace(pb, hids, hps, seed, sc_o, mode=1, max_steps=1000)
        for a, b in zip(a_all, b_all):
            same = (len(a) == len(b) and (a["region"] == b["region"]).all() and (a["ivox"] == b["ivox"]).all()
                    and (a["cause"] == b["cause"]).all())
            if same and float(np.abs(a["r"] - b["r"]).max()) <= DRIFT_MM:
                continue
            n_re += 0 if same else 1
            n_drift += 1 if same else 0
            for t, sign in ((a, +1.0), (b, -1.0)):
                ct = t["region"] == O.REG_CT
                iv = t["ivox"][ct].astype(np.int64)
                v = iv[:, 0] + n_xy[0] * (iv[:, 1] + n_xy[1] * iv[:, 2])
                np.add.at(delta, v, sign * t["dep"][ct].astype(np.float64))
                mask[v] = True
    return n_re, n_drift, delta, mask


def compare_row(O, pb, a_cv, b_dense, delta_edep, touched, nvox, rel_thr, hps):
    """A10(ii) for one row.  a_cv = the CUDA row (col, val); b_dense = the oracle's dense fp32 column; delta_edep = the
    energy the FLAGGED histories account for (their traced deposits, CUDA minus oracle, MeV), `touched` = the voxels they
    visit.  With pred = b_dense + dose(delta_edep) and tol_v = 2e-4 pred_v + dose_v(3 x DRIFT_MM x S_MAX x RSP_max) (what
    unflagged histories can move) + 1e-7 max (fp32 sums):
      * every kept value equals pred within tol;
      * the kept set equals {pred >= threshold} except for entries within 0.1 % of the threshold + tol;
      * outside the voxels of flagged histories pred IS the oracle's column, so there this is A10(ii) as written, up to
        the 0.01 um the unflagged histories may have moved.
    Returns (#one-sided entries at the threshold, #kept-set differences against the plain oracle row that the flagged
    histories explain)."""
    a = np.zeros(nvox, dtype=np.float64)
    a[a_cv[0]] = a_cv[1]
    b = b_dense.astype(np.float64)
    mx = b.max()
    if mx == 0.0:
        assert a.max() == 0.0
        return 0, 0
    pred = b + O.dose_from_edep(pb, delta_edep, 1.0 / hps)
    mxp = max(pred.max(), mx)
    thr = rel_thr * float(np.float32(a.max()))            # the CUDA row's own threshold (its column maximum is kept)
    tol = 2e-4 * np.abs(pred) + O.dose_from_edep(pb, np.full(nvox, 3.0 * DRIFT_MM * S_MAX * 2.5), 1.0 / hps) + 1e-7 * mxp
    kept = a > 0
    assert abs(a.max() - pred.max()) <= 2e-4 * mxp
    bad = kept & (np.abs(a - pred) > tol)
    assert not bad.any(), ("kept values differ from oracle + flagged histories", int(bad.sum()), np.flatnonzero(bad)[:5], a[bad][:5], pred[bad][:5])
    should = pred >= thr
    one = kept != should
    near = one & (np.abs(pred - thr) <= 1e-3 * thr + tol)
    assert not (one & ~near).any(), ("kept set differs away from the threshold", np.flatnonzero(one & ~near)[:5], pred[one & ~near][:5] / thr)
    thr_o = rel_thr * mx                                    # the plain oracle row's own threshold
    explained = (kept != ((b > 0) & (b >= thr_o))) & ~near
    # away from the flagged histories' voxels pred IS the oracle's value, so a difference there can only come from the
    # threshold itself: the flagged histories moved the column maximum, and the value lies between the two thresholds
    between = (b >= min(thr, thr_o) * (1.0 - 1e-3) - tol) & (b <= max(thr, thr_o) * (1.0 + 1e-3) + tol)
    assert not (explained & ~touched & ~between).any(), "a kept-set difference outside the voxels of flagged histories"
    assert abs(a.sum() - b[b >= rel_thr * mx].sum()) <= 2e-3 * b.sum()
    return int(near.sum()), int(explained.sum())


@pytest.mark.parametrize("n", [1, 7, 2047, 2048, 2049, 100003, 1 << 20])
def test_csr_writer_alone_is_bit_exact_on_synthetic_columns(bind, n):
    import torch
    O = orc()
    rng = np.random.default_rng(n)
    col = np.where(rng.random(n) < 0.3, rng.lognormal(0.0, 3.0, n), 0.0).astype(np.float32)
    if n > 10:
        col[5] = -1.0                                  # negative and exactly-at-threshold values
        col[7] = np.float32(1e-4) * col.max()
    eng = bind.Engine(wl.small_water())
    for thr in (1e-4, 0.0, 0.5):
        gi, gv = eng.csr_from_dense(torch.from_numpy(col).cuda(), thr)
        oi, ov = O.csr_row(col, thr)
        assert np.array_equal(gi.cpu().numpy(), oi) and np.array_equal(gv.cpu().numpy(), ov)
    z = torch.zeros(max(n, 1), dtype=torch.float32, device="cuda")
    gi, gv = eng.csr_from_dense(z, 1e-4)                # empty column -> empty row
    assert gi.numel() == 0 and gv.numel() == 0
    eng.close()


def test_csr_writer_alone_on_an_oracle_column(bind):
    import torch
    O = orc()
    w = hetero_case()
    pb = oracle_problem(w)
    col = O.influence_column(pb, 1, 3000, 5)
    eng = bind.Engine(w)
    gi, gv = eng.csr_from_dense(torch.from_numpy(col).cuda(), 1e-4)
    oi, ov = O.csr_row(col, 1e-4)
    assert oi.size > 100
    assert np.array_equal(gi.cpu().numpy(), oi) and np.array_equal(gv.cpu().numpy(), ov)
    eng.close()


SCEN = [((0.0, 0.0, 0.0), 1.0), ((3.0, 0.0, 0.0), 1.0), ((0.0, -3.0, 3.0), 1.035), ((0.0, 0.0, -3.0), 0.965)]


@pytest.mark.parametrize("case", ["hetero", "rs_ap", "rotated"])
def test_influence_parity(bind, case):
    O = orc()
    w = {"hetero": hetero_case, "rs_ap": rs_case, "rotated": rotated_case}[case]()
    hps, thr, seed = 10000, 1e-4, 9
    eng = bind.Engine(w)
    pb = oracle_problem(w)
    nvox = eng.nvox
    res = eng.influence([bind.scenario(s, k) for s, k in SCEN], hps, thr, seed)
    t = eng.tallies().as_dict()
    assert sum(t[k] for k in ("n_stopped_ct", "n_stopped_rs", "n_stopped_brass", "n_nuclear", "n_escaped")) == len(SCEN) * eng.n_spots * hps
    tot_near = tot_ex = tot_nnz = tot_re = tot_drift = 0
    for (shift, scale), (rp, col, val) in zip(SCEN, res):
        rp, col, val = rp.cpu().numpy(), col.cpu().numpy(), val.cpu().numpy()
        assert np.isfinite(val).all()
        check_csr_structure(rp, col, val, eng.n_spots, nvox)
        sc_o = O.scenario(shift, float(np.float32(scale)))
        sa = np.zeros(nvox); sb = np.zeros(nvox); sd = np.zeros(nvox)
        for g in range(eng.n_spots):
            b_dense = O.influence_column(pb, g, hps, seed, sc_o)
            n_re, n_drift, delta, touched = flagged_histories(bind, eng, O, pb, g, hps, seed, (shift, scale), nvox, eng.n[:2])
            near, ex = compare_row(O, pb, (col[rp[g]:rp[g + 1]], val[rp[g]:rp[g + 1]]), b_dense, delta, touched, nvox, thr, hps)
            tot_near += near; tot_ex += ex; tot_re += n_re; tot_drift += n_drift; tot_nnz += int(rp[g + 1] - rp[g])
            sa[col[rp[g]:rp[g + 1]]] += val[rp[g]:rp[g + 1]]; sb += b_dense
            sd += O.dose_from_edep(pb, delta, 1.0 / hps)
        err_sum = np.abs(sa - sb).max() / sb.max()
        err_acc = np.abs(sa - sb - sd).max() / sb.max()
        print(case, shift, scale, "sum of columns: max |d| / max = %.2e raw, %.2e with the flagged histories' own deposits accounted for" % (err_sum, err_acc))
        assert err_acc <= 2e-4 + thr * eng.n_spots            # entries below the threshold are missing from the CSR rows
        # raw bar of north_star (1e-3 of the maximum) where the 1-3 x 10^4 histories of the case allow it; behind the range
        # shifter f ~ 1e-2 of 2 x 10^4 histories are re-dealt: printed, bounded as a sanity check only
        assert err_sum <= (1e-3 if case != "rs_ap" else 5e-2)
    n_hist = len(SCEN) * eng.n_spots * hps
    print(case, "nnz", tot_nnz, "| histories", n_hist, "re-dealt", tot_re, "drifted >", DRIFT_MM, "mm:", tot_drift,
          "| one-sided entries at the threshold", tot_near, "| kept-set differences explained by flagged histories", tot_ex)
    assert tot_nnz > 1000
    # sanity bounds only: how many histories two fp32 / fp64 implementations of this method re-deal is a property of the
    # method (tests/test_method_sensitivity.py); the numbers are printed above and recorded in profiles/
    assert tot_re <= (3e-2 if case == "rs_ap" else 5e-3) * n_hist
    eng.close()


def test_influence_groups_and_replay_give_the_same_matrix(bind):
    """Small workspace -> several groups; zero box margin -> the overflow list, or without it the replay path; all must
    reproduce the default run."""
    w = hetero_case()
    hps, thr, seed = 3000, 1e-4, 3
    sc = [bind.scenario((0, 0, 0), 1.0)]
    eng = bind.Engine(w)
    eng.set_timing(True)

    def run():
        eng.timing()
        m = [x.cpu().numpy() for x in eng.influence(sc, hps, thr, seed)[0]]
        return m, eng.timing()["voxel"][1]              # passes of the pipeline: pilot + groups (+ replays)

    base, p_base = run()
    eng.set_workspace_limit(4 * 1024)                   # 1024 box elements: one column per group
    small, p_small = run()
    eng.set_knob(bind.KNOB_BOX_GROW, 0); eng.set_knob(bind.KNOB_BOX_PAD, 0)
    eng.set_workspace_limit(0)
    overflow, p_ovf = run()                             # tight boxes: the overflow list fills the rows
    eng.set_knob(bind.KNOB_OVF_CAP, 0)                  # no list: the replay path
    replay, p_replay = run()
    eng.set_knob(bind.KNOB_OVF_CAP, 1 << 25); eng.set_knob(bind.KNOB_OVF_SORT_CAP, 8)      # a list, but buckets of more than 8 entries
    bucket, p_bucket = run()                            # per column are not sorted: those columns are replayed with a larger box
    eng.set_knob(bind.KNOB_OVF_SORT_CAP, 16384)
    assert p_base == 2 and p_small == 1 + eng.n_spots and p_ovf == 2 and p_replay == 3 and p_bucket >= 3, (p_base, p_small, p_ovf, p_replay, p_bucket)
    # the same histories in another launch order: identical structure up to entries at the threshold, values to fp32 sums
    none = np.zeros(eng.nvox, dtype=bool); zero = np.zeros(eng.nvox)
    for other in (small, overflow, replay, bucket):
        check_csr_structure(*other, eng.n_spots, eng.nvox)
        for g in range(eng.n_spots):
            dense = np.zeros(eng.nvox, dtype=np.float32)
            dense[base[1][base[0][g]:base[0][g + 1]]] = base[2][base[0][g]:base[0][g + 1]]
            lo, hi = other[0][g], other[0][g + 1]
            a = np.zeros(eng.nvox); a[other[1][lo:hi]] = other[2][lo:hi]
            both = (a > 0) & (dense > 0)
            assert np.abs(a - dense)[both].max() <= 1e-5 * dense.max()
            one = (a > 0) != (dense > 0)
            assert (np.abs(np.maximum(a, dense)[one] - thr * dense.max()) <= 1e-3 * thr * dense.max()).all()
    eng.close()


def test_nominal_influence_column_equals_dose_of_the_same_histories(bind):
    """One spot, N = hist_per_spot: dose-mode ids and influence-mode ids coincide, so dose = weight * column (C1, C2)."""
    w = wl.small_water(n=(20, 20, 40), energy=80.0, sigma=3.0, n_spots=1, with_aperture=True, opening_radius=4.0)
    w["beams"][0]["spots"][0, 3] = 2.5                 # weight
    N, seed = 20000, 4
    eng = bind.Engine(w, bind.default_params(n_batches=1))
    d = eng.dose(N, seed).cpu().numpy().astype(np.float64)
    rp, col, val = [x.cpu().numpy() for x in eng.influence([bind.scenario()], N, 0.0, seed)[0]]
    dense = np.zeros(eng.nvox); dense[col] = val
    assert rp[1] == col.size == int((d > 0).sum())
    assert np.abs(2.5 * dense - d).max() <= 1e-5 * d.max()      # fp32 scale factors and atomic order
    eng.close()


def test_influence_edge_cases(bind):
    # a spot that is fully absorbed in a closed block gives an empty row; hist_per_spot = 1 works
    w = wl.small_water(n=(20, 20, 30), energy=120.0, sigma=2.0, with_aperture=True, n_spots=2)
    w["beams"][0]["aperture"]["open"][:] = 0
    eng = bind.Engine(w)
    rp, col, val = eng.influence([bind.scenario()], 500, 1e-4, 1)[0]
    assert rp.cpu().numpy().tolist() == [0, 0, 0] and col.numel() == 0
    eng.close()
    eng = bind.Engine(wl.small_water(n_spots=3))
    rp, col, val = eng.influence([bind.scenario()], 1, 1e-4, 1)[0]
    check_csr_structure(rp.cpu().numpy(), col.cpu().numpy(), val.cpu().numpy(), 3, eng.nvox)
    with pytest.raises(bind.VpmcError):
        eng.influence([bind.scenario(rsp_scale=0.0)], 10, 1e-4, 1)
    eng.close()
