"""SURVEY.md 8(f)-3, second half: the 3-D gamma index on the device (vpmc_gamma) against the oracle's tool
(oracle/vpmc_oracle.py gamma_counts, itself pinned by tests/test_oracle_geometry.py::test_gamma_tool).  The number of voxels
evaluated is an integer of the inputs and must be equal; a voxel's pass / fail is a floating-point decision taken in fp32
on the device and fp64 in the oracle, so voxels whose minimum gamma^2 lies within 1e-5 of 1 may differ: none is expected on
these cases and at most 2 are allowed."""
import numpy as np
import pytest
import torch

from paper_2307_01416_b200 import workloads as wl
from tests.helpers import grid, oracle_problem

pytestmark = pytest.mark.gpu


def _blob(n, h, centre, sigma, amp=1.0):
    z, y, x = np.meshgrid(*[(np.arange(k) + 0.5) * s for k, s in zip(n[::-1], h[::-1])], indexing="ij")
    r2 = (x - centre[0]) ** 2 + (y - centre[1]) ** 2 + (z - centre[2]) ** 2
    return (amp * np.exp(-r2 / (2 * sigma ** 2))).astype(np.float32)


def _engine(n, h):
    from paper_2307_01416_b200 import binding
    w = wl.small_water(n=n, h=h)
    return binding.Engine(w), w


@pytest.mark.parametrize("h", [(1.0, 1.0, 1.0), (1.0, 1.0, 1.5), (2.0, 2.5, 1.5)])
def test_gamma_counts_match_the_oracle_on_synthetic_grids(h):
    from oracle import vpmc_oracle as O
    n = (40, 36, 30)
    eng, w = _engine(n, h)
    ext = [k * s for k, s in zip(n, h)]
    c = [0.5 * e for e in ext]
    ref = _blob(n, h, c, 8.0)
    rng = np.random.default_rng(1)
    cases = {
        "same": ref.copy(),
        "scaled_in": ref * np.float32(1.005),
        "scaled_out": ref * np.float32(1.2),
        "shift_half_mm": _blob(n, h, (c[0] + 0.5, c[1], c[2]), 8.0),
        "shift_far": _blob(n, h, (c[0] + 4.0, c[1] - 3.0, c[2]), 8.0),
        "noisy": (ref * (1.0 + 0.02 * rng.standard_normal(ref.shape))).astype(np.float32),
        "corner": _blob(n, h, (1.0, 1.0, 1.0), 6.0) * np.float32(1.03),          # hot voxels on the grid's edge: clamped lookups
    }
    refs = {"corner": _blob(n, h, (1.3, 0.8, 1.0), 6.0)}
    for name, ev in cases.items():
        r = refs.get(name, ref)
        ne_o, nf_o = O.gamma_counts(r, ev, h, dd=0.01, dta=1.0, thr=0.1)
        rate, ne, nf = eng.gamma(torch.from_numpy(r.reshape(-1)).cuda(), torch.from_numpy(ev.reshape(-1)).cuda(), 0.01, 1.0, 0.1)
        print(h, name, "evaluated", ne, "failing gpu", nf, "oracle", nf_o)
        assert ne == ne_o and ne > 0
        assert abs(nf - nf_o) <= 2, (name, nf, nf_o)
        assert abs(rate - (1.0 - nf_o / ne_o)) <= 2.0 / ne_o
    # other criteria (Table 2 of the paper uses 2 %/2 mm and 3 %/3 mm as well)
    ev = cases["shift_far"]
    for dd, dta in ((0.02, 2.0), (0.03, 3.0)):
        ne_o, nf_o = O.gamma_counts(ref, ev, h, dd=dd, dta=dta, thr=0.1, sub=5)
        _, ne, nf = eng.gamma(torch.from_numpy(ref.reshape(-1)).cuda(), torch.from_numpy(ev.reshape(-1)).cuda(), dd, dta, 0.1, sub=5)
        assert ne == ne_o and abs(nf - nf_o) <= 2
    eng.close()


def test_gamma_of_a_transported_dose_against_the_oracle_dose():
    """The use the tests make of it: the GPU dose of config 1 against the oracle dose, gamma 1 %/1 mm/10 % >= 99.9 % -- computed by
    the device kernel and by the oracle's tool on the same two grids."""
    from paper_2307_01416_b200 import binding
    from oracle import vpmc_oracle as O
    w = wl.config1()
    eng = binding.Engine(w)
    N, seed = 100_000, 1
    d_gpu = eng.dose(N, seed)
    d_orc, _ = O.dose(oracle_problem(w), N, seed)
    ref32 = d_orc.astype(np.float32)
    rate, ne, nf = eng.gamma(torch.from_numpy(ref32).cuda(), d_gpu, 0.01, 1.0, 0.1)
    ne_o, nf_o = O.gamma_counts(grid(w, ref32), grid(w, d_gpu.cpu().numpy()), w["ct"]["h"], 0.01, 1.0, 0.1)
    assert ne == ne_o and abs(nf - nf_o) <= 2 and rate >= 0.999
    # and a deliberately wrong dose fails (x 1.5: at 10^5 histories the voxel-to-voxel noise lets a 10 % error find a match within 1 mm)
    wrong = (d_gpu * 1.5).contiguous()
    rate2, _, nf2 = eng.gamma(torch.from_numpy(ref32).cuda(), wrong, 0.01, 1.0, 0.1)
    ne3, nf3 = O.gamma_counts(grid(w, ref32), grid(w, wrong.cpu().numpy()), w["ct"]["h"], 0.01, 1.0, 0.1)
    assert rate2 < 0.5 and abs(nf2 - nf3) <= 2
    eng.close()
