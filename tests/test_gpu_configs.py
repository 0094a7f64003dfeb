"""GPU parity at the sizes of BASELINE.json configs 2-5, in the launch configuration bench.py times.

At these sizes the oracle cannot run the whole job, so parity is checked on WINDOWS of 10^6 history ids
of the full-size run -- exact, because Philox streams are keyed by history id -- with the bar north_star states (1e-3 of the
maximum dose, gamma 1 % / 1 mm >= 99.9 %), and on properties that hold at any size (bookkeeping, counts, integral dose)."""
import numpy as np
import pytest

from paper_2307_01416_b200 import workloads as wl
from tests.helpers import grid, oracle_columns_parallel, oracle_problem, oracle_window_parallel

pytestmark = pytest.mark.gpu
COUNTS = ("n_stopped_ct", "n_stopped_rs", "n_stopped_brass", "n_nuclear", "n_escaped")


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


WINDOW = 1_000_000          # parity prefixes of >= 10^6 history ids
DRIFT_MM = 1e-4             # end-point difference above which a history counts as drifted (0.1 um)


def traced_deposits(O, traces, n_xy, nvox, gamma_loc, sign, out):
    for t in traces:
        ct = t["region"] == O.REG_CT
        iv = t["ivox"][ct].astype(np.int64)
        v = iv[:, 0] + n_xy[0] * (iv[:, 1] + n_xy[1] * iv[:, 2])
        np.add.at(out, v, sign * t["dep"][ct].astype(np.float64))


def window_parity(bind, fn, kw, seed, lo, sc=None, n_ids=WINDOW, raw_bar=True):
    """History ids [lo, lo + n_ids) of the full-size run on the GPU (bench.py's launch configuration) against the oracle on
    the same ids (the single-threaded oracle, one process per host core on disjoint id ranges).

    Two implementations of this method that differ in the last bit cannot agree on every history: at a
    near-tie a history changes its voxel sequence and its later deflections are re-dealt, and the differences of the
    others grow along the path.  So the comparison is made in two parts that together account for EVERY voxel:
      1. per-history digests (number of records, hash of the discrete trace, end point) of all ids on both sides find the
         FLAGGED histories: discrete trace differs (re-dealt), or end point moved by more than DRIFT_MM (drifted).  Their
         numbers are printed; how many there are is a property of the method, not of the arithmetic type (the oracle
         re-deals as many of its own histories when one constant moves by 1e-6: tests/test_method_sensitivity.py);
      2. with the flagged histories' own traced deposits (CUDA minus oracle) added to the oracle's grid, the production
         dose must equal it to 2e-4 of the maximum dose in EVERY voxel: all other histories, the scoring and the dose
         conversion agree five times better than north_star's 1e-3.
    The raw bar (max |dD| <= 1e-3 D_max, gamma 1 % / 1 mm / 10 % >= 99.9 %, no correction) is asserted as well where the
    run holds enough histories per voxel (raw_bar), and printed otherwise: a re-dealt fraction f shifts a voxel by
    sqrt(2 f) of its own statistical error, i.e. by 7e-4 of the local dose once the plan is run to the 0.5 % uncertainty
    of the metric (f = 1e-2)."""
    O = orc()
    w = getattr(wl, fn)(**kw)
    N = w["n_histories"]
    hi = lo + n_ids
    scg = None if sc is None else bind.scenario(*sc)
    sco = None if sc is None else O.scenario(sc[0], float(np.float32(sc[1])))
    eng = bind.Engine(w, bind.default_params(n_batches=1))
    eng.set_history_window(lo, hi)
    d_gpu = eng.dose(N, seed, sc=scg).cpu().numpy().astype(np.float64)
    tg = eng.tallies().as_dict()
    eng.set_history_window(0, 0)
    dg = eng.digests(N, seed, lo, n_ids, sc=scg)
    assert np.isfinite(d_gpu).all()
    pb = oracle_problem(w)
    e, to, do = oracle_window_parallel(fn, kw, pb.nvox, N, seed, lo, hi, sc, digests=True)
    d_orc = O.dose_from_edep(pb, e, pb.total_weight / N)
    mx = d_orc.max()
    assert mx > 0
    # ---- 1. flagged histories
    assert (dg["hid"] == do["hid"]).all()
    redealt = (dg["hash"] != do["hash"]) | (dg["n_rec"] != do["n_rec"]) | (dg["cause"] != do["cause"])
    drifted = ~redealt & (np.abs(dg["r"].astype(np.float64) - do["r"]).max(axis=1) > DRIFT_MM)
    flagged = np.flatnonzero(redealt | drifted)
    delta = np.zeros(pb.nvox, dtype=np.float64)
    n_xy = w["ct"]["n"][:2]
    for i0 in range(0, flagged.size, 2500):
        hids = dg["hid"][flagged[i0:i0 + 2500]]
        traced_deposits(O, eng.trace(hids, N, seed, sc=scg, max_steps=1200), n_xy, pb.nvox, float(pb.params.gamma_loc), +1.0, delta)
        traced_deposits(O, O.trace(pb, hids, N, seed, sco, max_steps=1200), n_xy, pb.nvox, float(pb.params.gamma_loc), -1.0, delta)
    eng.close()
    # ---- 2. everything else
    pred = d_orc + O.dose_from_edep(pb, delta, pb.total_weight / N)
    err_rest = np.abs(d_gpu - pred).max() / mx
    err_raw = np.abs(d_gpu - d_orc).max() / mx
    gam = O.gamma_pass_rate(grid(w, d_orc), grid(w, d_gpu), w["ct"]["h"], dd=0.01, dta=1.0, thr=0.1)
    f = flagged.size / n_ids
    print(w["name"], "window", lo, hi, "| flagged %.4f (re-dealt %d, drifted > %g mm %d)" % (f, int(redealt.sum()), DRIFT_MM, int(drifted.sum())),
          "| all other histories + scoring: max |dD|/Dmax = %.2e" % err_rest, "| raw: max |dD|/Dmax = %.3e, gamma 1%%/1mm = %.5f" % (err_raw, gam),
          "| counts gpu", [tg[k] for k in COUNTS], "orc", [to[k] for k in COUNTS])
    assert int(redealt.sum()) <= 0.25 * n_ids            # sanity only, see the docstring
    assert err_rest <= 2e-4
    if raw_bar:
        assert err_raw <= 1e-3
        assert gam >= 0.999
    assert sum(tg[k] for k in COUNTS) == hi - lo
    for k in COUNTS:
        assert abs(int(tg[k]) - int(to[k])) <= max(3, 1e-4 * (hi - lo)), k
    for k in ("incident", "dep_ct", "dep_rs", "dep_brass", "escaped", "removed"):
        assert abs(tg[k] - to[k]) <= 2e-5 * to["incident"], (k, tg[k], to[k])


def test_config2_full_size_properties_and_window(bind):
    """10^7 histories of a config-2 plan (range shifter, 2 cm opening), exactly as bench.py launches it."""
    w = wl.config2(20, True)
    N = w["n_histories"]
    eng = bind.Engine(w)
    d = eng.dose(N, 2)
    t = eng.tallies().as_dict()
    u = eng.uncertainty()
    assert sum(t[k] for k in COUNTS) == N
    total = t["dep_ct"] + t["dep_rs"] + t["dep_brass"] + t["escaped"] + t["removed"]
    assert abs(total - t["incident"]) <= 1e-6 * t["incident"]
    cnt = orc().spot_counts(oracle_problem(w), N).astype(np.float64)          # C2 apportionment (integer-exact)
    assert cnt.sum() == N
    assert abs(t["incident"] - float((cnt * w["beams"][0]["spots"][:, 2].astype(np.float64)).sum())) <= 1e-9 * t["incident"]
    assert t["n_stopped_rs"] > 0 and t["n_stopped_brass"] > 0.5 * N          # 70 / 72.5 MeV stop in the slab (P9), brass absorbs (P7)
    # integral: sum_v D_v rho_v V = (W/N) dep_ct 1.602e-10 / 1e-3   (water: rho = 1, V = 8e-3 cm^3)
    W = float(w["beams"][0]["spots"][:, 3].sum())
    assert abs(float(d.double().sum()) * 8e-3 / 1.602176634e-10 - W / N * t["dep_ct"]) <= 1e-4 * W / N * t["dep_ct"]
    assert 0.0 < u < 0.02
    eng.close()
    assert np.isfinite(d.cpu().numpy()).all()
    window_parity(bind, "config2", {"opening_mm": 20, "range_shifter": True}, 2, 4_500_000, raw_bar=False)
    # the raw bar on the WHOLE 10^7-history plan (the oracle over all host cores)
    O = orc()
    pb = oracle_problem(w)
    e, to = oracle_window_parallel("config2", {"opening_mm": 20, "range_shifter": True}, pb.nvox, N, 2, 0, N)
    d_orc = O.dose_from_edep(pb, e, pb.total_weight / N)
    d_gpu = d.cpu().numpy().astype(np.float64)
    err = np.abs(d_gpu - d_orc).max() / d_orc.max()
    gam = O.gamma_pass_rate(grid(w, d_orc), grid(w, d_gpu), w["ct"]["h"], dd=0.01, dta=1.0, thr=0.1)
    print("config2 whole plan, 10^7 histories: max |dD|/Dmax = %.3e, gamma 1%%/1mm = %.5f" % (err, gam), "counts gpu", [t[k] for k in COUNTS], "orc", [to[k] for k in COUNTS])
    assert err <= 1e-3 and gam >= 0.999
    for k in COUNTS:
        assert abs(int(t[k]) - int(to[k])) <= 1e-4 * N, k


def test_config3_head_window(bind):
    # 1 x 1 x 1.5 mm voxels, ~6000 spots: a 10^6-id window puts tens of histories into a voxel, and a history that stops
    # in an air voxel (rho 0.0012) alone makes a dose of 0.8 D_max there: the raw per-voxel bar is printed, not asserted
    window_parity(bind, "config3", {"seed": 3}, 3, 2_000_000, raw_bar=False)
    window_parity(bind, "config3", {"seed": 3}, 3, 7_500_000, sc=((0.0, 3.0, -3.0), 0.965), raw_bar=False)


def test_config3_trace(bind):
    O = orc()
    w = wl.config3(3)
    N = 10_000_000
    eng = bind.Engine(w)
    hids = np.arange(1024, dtype=np.uint64) * (N // 1024)
    g = eng.trace(hids, N, 3, max_steps=900)
    o = O.trace(oracle_problem(w), hids, N, 3, max_steps=900)
    eng.close()
    errs, nd = [], 0
    for a, b in zip(g, o):
        if not (len(a) == len(b) and (a["region"] == b["region"]).all() and (a["ivox"] == b["ivox"]).all() and (a["cause"] == b["cause"]).all()):
            nd += 1
            continue
        errs.append(max(float(np.abs(a["E_after"] - b["E_after"]).max()) / float(b["E_before"][0]),
                        float(np.abs(a["r"] - b["r"]).max()) / 256.0, float(np.abs(a["u"] - b["u"]).max())))
    errs = np.array(errs)
    print("config3 trace: mismatches", nd, "of 1024, median %.2e p99 %.2e" % (np.median(errs), np.quantile(errs, 0.99)))
    assert nd <= 16 and np.median(errs) < 5e-6


def test_config5_stress_window(bind):
    # ids of the central spots of the 170 MeV layer (spot 40 * 121 + 60 of 7865, ~12714 histories each)
    # 1 mm voxels, range shifter: ~40 histories in the hottest voxel of a 10^6-id window (raw bar printed, not asserted)
    window_parity(bind, "config5", {}, 5, 62_000_000, raw_bar=False)


def test_config4_influence_13_scenarios(bind):
    """The full spot list (~2000 spots, 2 beams) under the 13 scenarios at the config's 10^4 histories per spot; 8 rows
    of 4 scenarios against the oracle with A10(ii) as written (tests/test_gpu_influence.py)."""
    from tests.test_gpu_influence import DRIFT_MM as DRIFT_INF, compare_row, flagged_histories
    O = orc()
    w = wl.config4()
    hps, thr, seed = w["hist_per_spot"], 1e-4, 4
    assert hps == 10_000
    eng = bind.Engine(w)
    ns = eng.n_spots
    assert 1800 <= ns <= 2200 and len(w["scenarios"]) == 13
    res = eng.influence([bind.scenario(s, k) for s, k in w["scenarios"]], hps, thr, seed)
    t = eng.tallies().as_dict()
    assert sum(t[k] for k in COUNTS) == 13 * ns * hps
    pb = oracle_problem(w)
    rows = [0, ns // 7, 2 * ns // 7, 3 * ns // 7, ns // 2, 5 * ns // 7, 6 * ns // 7, ns - 1]
    nnz_tot = n_near = n_ex = n_re = n_drift = 0
    for si, (rp, col, val) in enumerate(res):
        rp, col, val = rp.cpu().numpy(), col.cpu().numpy(), val.cpu().numpy()
        assert rp.shape == (ns + 1,) and rp[0] == 0 and (np.diff(rp) >= 0).all() and rp[-1] == col.size == val.size
        assert np.isfinite(val).all() and (val > 0).all() and col.min() >= 0 and col.max() < eng.nvox
        nnz_tot += col.size
        if si in (0, 3, 8, 11):                          # nominal, -y shift, range -3.5 %, (range +3.5 %, z -3 mm)
            shift, scale = w["scenarios"][si]
            cols = oracle_columns_parallel("config4", {}, pb.nvox, rows, hps, seed, (shift, scale))
            for g, e in zip(rows, cols):
                c = col[rp[g]:rp[g + 1]]; v = val[rp[g]:rp[g + 1]]
                assert (np.diff(c) > 0).all()
                b_dense = O.dose_from_edep(pb, e, 1.0 / hps).astype(np.float32)
                re, drift, delta, touched = flagged_histories(bind, eng, O, pb, g, hps, seed, (shift, scale), eng.nvox, eng.n[:2])
                near, ex = compare_row(O, pb, (c, v), b_dense, delta, touched, eng.nvox, thr, hps)
                n_near += near; n_ex += ex; n_re += re; n_drift += drift
    print("config4: spots", ns, "nnz over 13 scenarios", nnz_tot, "launches", eng.launch_count(), "| 32 columns checked:", 32 * hps, "histories, re-dealt",
          n_re, "drifted >", DRIFT_INF, "mm:", n_drift, "| one-sided entries at the threshold", n_near, "| kept-set differences explained by flagged histories", n_ex)
    assert n_re <= 1.5e-2 * 32 * hps
    eng.close()
