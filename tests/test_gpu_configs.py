"""GPU parity at the sizes of BASELINE.json configs 2-5, in the launch configuration bench.py times.

At these sizes the single-threaded oracle cannot run the whole job, so parity is checked on WINDOWS of
history ids of the full-size run -- exact, because Philox streams are keyed by history id -- and on properties that hold
at any size (bookkeeping, counts, integral dose).  A window of 2e4 histories spread over 1 mm voxels puts only tens of
histories into a voxel, so the per-voxel bar is the one DESIGN.md 4.2 derives: identical histories give identical
deposits (the bulk of the voxels agree to 1e-3 of the maximum), a re-dealt history moves its own deposits."""
import numpy as np
import pytest

from paper_2307_01416_b200 import workloads as wl
from tests.helpers import oracle_problem

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


def window_parity(bind, w, N, seed, lo, hi, sc=None, frac_ok=0.995, slice_tol=5e-3):
    O = orc()
    eng = bind.Engine(w, bind.default_params(n_batches=1))
    eng.set_history_window(lo, hi)
    d_gpu = eng.dose(N, seed, sc=None if sc is None else bind.scenario(*sc)).cpu().numpy().astype(np.float64)
    tg = eng.tallies().as_dict()
    eng.close()
    pb = oracle_problem(w)
    e, to = O.dose_edep(pb, N, seed, None if sc is None else O.scenario(sc[0], float(np.float32(sc[1]))), hid_begin=lo, hid_end=hi)
    d_orc = O.dose_from_edep(pb, e, pb.total_weight / N)
    to = to.as_dict()
    mx = d_orc.max()
    assert mx > 0
    nz = (d_orc > 0) | (d_gpu > 0)
    dev = np.abs(d_gpu - d_orc)[nz] / mx
    print(w["name"], "window", lo, hi, "voxels", int(nz.sum()), "within 1e-3: %.5f" % np.mean(dev <= 1e-3), "max %.3e" % dev.max(),
          "counts gpu", [tg[k] for k in COUNTS], "orc", [to[k] for k in COUNTS])
    assert np.mean(dev <= 1e-3) >= frac_ok
    assert sum(tg[k] for k in COUNTS) == hi - lo
    for k in COUNTS:
        assert abs(int(tg[k]) - int(to[k])) <= max(3, 2e-3 * (hi - lo)), k
    for k in ("incident", "dep_ct", "dep_rs", "dep_brass", "escaped", "removed"):
        assert abs(tg[k] - to[k]) <= 1e-4 * to["incident"], (k, tg[k], to[k])
    # integral dose, in all and per z-slice (a re-dealt history moves its deposits sideways, hardly in depth)
    assert abs(d_gpu.sum() - d_orc.sum()) <= 5e-3 * d_orc.sum()
    nz_ = w["ct"]["n"][2]
    sg, so = d_gpu.reshape(nz_, -1).sum(1), d_orc.reshape(nz_, -1).sum(1)
    big = so >= 0.05 * so.max()
    assert np.abs(sg[big] / so[big] - 1.0).max() <= slice_tol, np.abs(sg[big] / so[big] - 1.0).max()


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
    window_parity(bind, w, N, 2, 5_000_000, 5_020_000, frac_ok=0.98)      # 1.6 spots only: few voxels, each re-dealt history shows


def test_config3_head_window(bind):
    w = wl.config3(3)
    window_parity(bind, w, 10_000_000, 3, 2_000_000, 2_020_000)
    window_parity(bind, w, 10_000_000, 3, 7_500_000, 7_520_000, sc=((0.0, 3.0, -3.0), 0.965))


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
    w = wl.config5()
    # ids of the central spots of the 170 MeV layer (spot 40*121 + 60 of 7865, ~12714 histories each)
    # 170 steps through 1 mm voxels with about ONE history per voxel: every re-dealt history shows in the
    # voxels it touches (measured: 86 % of the voxels within 1e-3 of the maximum, termination counts identical, energy per
    # z-slice within 4e-3), so the per-voxel bar is loose here and the slice integrals carry the comparison
    window_parity(bind, w, w["n_histories"], 5, 62_300_000, 62_320_000, frac_ok=0.80, slice_tol=1e-2)


def test_config4_influence_13_scenarios(bind):
    """The full spot list (~2000 spots, 2 beams) under the 13 scenarios with few histories per spot; selected rows
    against the oracle."""
    O = orc()
    w = wl.config4()
    hps, thr, seed = 400, 1e-4, 4
    eng = bind.Engine(w)
    assert 1800 <= eng.n_spots <= 2200 and len(w["scenarios"]) == 13
    res = eng.influence([bind.scenario(s, k) for s, k in w["scenarios"]], hps, thr, seed)
    t = eng.tallies().as_dict()
    assert sum(t[k] for k in COUNTS) == 13 * eng.n_spots * hps
    pb = oracle_problem(w)
    nnz_tot = 0
    for si, (rp, col, val) in enumerate(res):
        rp, col, val = rp.cpu().numpy(), col.cpu().numpy(), val.cpu().numpy()
        assert rp.shape == (eng.n_spots + 1,) and rp[0] == 0 and (np.diff(rp) >= 0).all() and rp[-1] == col.size == val.size
        assert (val > 0).all() and col.min() >= 0 and col.max() < eng.nvox
        nnz_tot += col.size
        if si in (0, 9):
            shift, scale = w["scenarios"][si]
            for g in (0, eng.n_spots // 2, eng.n_spots - 1):
                c = col[rp[g]:rp[g + 1]]; v = val[rp[g]:rp[g + 1]]
                assert (np.diff(c) > 0).all()
                oc, ov = O.csr_row(O.influence_column(pb, g, hps, seed, O.scenario(shift, float(np.float32(scale)))), thr)
                a = np.zeros(eng.nvox); a[c] = v
                b = np.zeros(eng.nvox); b[oc] = ov
                assert abs(a.sum() - b.sum()) <= 5e-3 * b.sum()
                both = (a > 0) & (b > 0)
                assert np.mean(np.abs(a[both] - b[both]) <= 1e-3 * b.max()) >= 0.95
                assert abs(int((a > 0).sum()) - int((b > 0).sum())) <= 0.03 * (b > 0).sum()
    print("config4: spots", eng.n_spots, "nnz over 13 scenarios", nnz_tot, "launches", eng.launch_count())
    eng.close()
