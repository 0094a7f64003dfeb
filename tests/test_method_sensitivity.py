"""How many histories the METHOD re-deals when its arithmetic changes in the seventh digit -- measured
with the oracle alone, no CUDA path involved.

C4 deals one Philox block per step and splits steps at voxel faces, so a position difference delta becomes a step-length
difference delta / |u_lateral| at a glancing face crossing, the two part-steps get other deflections, and the difference
grows by an order of magnitude per crossing; at a corner near-tie the voxel sequence changes and every later deflection is
re-dealt.  Two faithful implementations that differ in the last bits therefore disagree on a share of the histories that
depends on the workload (voxel size, path length, angular spread), not on which of them is "right".  This test pins that
share for the oracle against ITSELF with the three radiation lengths moved by 1e-6 relative (= every theta0 by 5e-7, eight
fp32 ulp): it is the yardstick the GPU parity tests print their own numbers against (tests/test_gpu_configs.py).
"""
import numpy as np

from oracle import vpmc_oracle as orc
from paper_2307_01416_b200 import workloads as wl
from tests.helpers import oracle_problem


def sensitivity(w, N, lo, n, eps, seed=3):
    base = orc.digests(oracle_problem(w), N, seed, lo, n)
    p = orc.params_as_f32(orc.default_params())
    p.X0_w *= 1 + eps; p.rs_X0 *= 1 + eps; p.brass_X0 *= 1 + eps
    d = orc.digests(orc.Problem(ct=w["ct"], calib=w["calib"], beams=w["beams"], params=p), N, seed, lo, n)
    re = (d["hash"] != base["hash"]) | (d["n_rec"] != base["n_rec"])
    dr = np.abs(d["r"] - base["r"]).max(axis=1)
    return float(re.mean()), float((~re & (dr > 1e-4)).mean()), float(np.median(dr[~re]))


def test_digest_is_deterministic_and_sees_a_changed_trace():
    w = wl.config1()
    pb = oracle_problem(w)
    a = orc.digests(pb, 100000, 1, 500, 64)
    b = orc.digests(pb, 100000, 1, 500, 64)
    assert np.array_equal(a, b)
    assert len(set(a["hash"].tolist())) >= 32                     # histories that stay in one voxel column share a trace
    r = orc.trace(pb, [503], 100000, 1)[0]
    assert a[3]["n_rec"] == len(r) and a[3]["cause"] == r[-1]["cause"] and np.allclose(a[3]["r"], r[-1]["r"], atol=0)
    c = orc.digests(pb, 100000, 2, 500, 64)                       # another seed: other traces
    assert (c["hash"] != a["hash"]).mean() > 0.5


def test_one_millimetre_voxels_behind_a_range_shifter_are_chaotic():
    """Config 5 (1 mm voxels, 45 mm range shifter, ~150 voxel layers): a 1e-6 change of the radiation lengths re-deals
    about one history in ten and moves the end point of a third of the others by more than 0.1 um."""
    re, drift, med = sensitivity(wl.config5(), 100_000_000, 62_000_000, 4000, 1e-6)
    print("config5: re-dealt %.4f, drifted > 0.1 um %.4f, median drift %.2e mm" % (re, drift, med))
    assert 0.05 < re < 0.25 and drift > 0.15
    re7, drift7, _ = sensitivity(wl.config5(), 100_000_000, 62_000_000, 4000, 1e-7)
    assert 0.01 < re7 < re                                         # ten times less perturbation: still a few per cent


def test_two_millimetre_water_is_not():
    """Config 2 (2 mm voxels, water): the same perturbation re-deals fewer than one history in a thousand."""
    re, drift, med = sensitivity(wl.config2(20, True), 10_000_000, 4_500_000, 4000, 1e-6)
    print("config2 rs: re-dealt %.4f, drifted > 0.1 um %.4f, median drift %.2e mm" % (re, drift, med))
    assert re < 2e-3 and drift < 0.02
