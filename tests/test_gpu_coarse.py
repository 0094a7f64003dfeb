"""SURVEY.md 8(f)-4 on the GPU: scoring on cells of several voxels (vpmc_set_scoring_grid) against the oracle's definition
(dose_from_edep_coarse on the oracle's own per-voxel E_dep): dose grids, the stopping-rule path, gamma on the scoring grid and
the influence matrices' cell columns."""
import numpy as np
import pytest
import torch

from paper_2307_01416_b200 import workloads as wl
from tests.helpers import oracle_problem
from tests.test_gpu_parity import hetero_case

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("div", [(2, 2, 2), (3, 1, 4), (5, 7, 3)])
def test_coarse_dose_against_the_oracle(div):
    from paper_2307_01416_b200 import binding
    from oracle import vpmc_oracle as O
    w = hetero_case()                                  # 24 x 20 x 40 voxels of 2 x 2.5 x 1.5 mm: ragged for (5, 7, 3)
    N, seed = 100_000, 1
    eng = binding.Engine(w)
    fine = eng.dose(N, seed).clone()
    sn = eng.set_scoring_grid(div)
    assert sn == tuple((n + d - 1) // d for n, d in zip(w["ct"]["n"], div)) and eng.ncell == sn[0] * sn[1] * sn[2]
    d_gpu = eng.dose(N, seed).cpu().numpy().astype(np.float64)
    unc = eng.uncertainty()
    pb = oracle_problem(w)
    e, _ = O.dose_edep(pb, N, seed)
    d_orc = O.dose_from_edep_coarse(pb, e, pb.total_weight / N, div)
    assert d_gpu.shape == d_orc.shape and np.isfinite(d_gpu).all()
    assert np.abs(d_gpu - d_orc).max() <= 1e-3 * d_orc.max()
    assert 0 < unc < 0.2
    # the GPU's own fine dose aggregated by the definition gives the same grid (same histories, another scoring index)
    cell, _ = O.coarse_cells(pb, div)
    hu = np.asarray(w["ct"]["hu"], dtype=np.float64).reshape(-1)
    rho = np.maximum(np.interp(hu, w["calib"]["hu"], w["calib"]["rho"]), float(pb.params.rho_min))
    agg = np.bincount(cell, weights=fine.cpu().numpy().astype(np.float64) * rho) / np.bincount(cell, weights=rho)
    assert np.abs(d_gpu - agg).max() <= 2e-5 * agg.max()
    # the device stopping rule and gamma run on the scoring grid
    out = eng.dose_to_uncertainty(20_000, 0.0, seed, min_batches=2, max_batches=3)
    assert out.numel() == eng.ncell and eng.run_info()[0] == 3
    rate, ne, nf = eng.gamma(torch.from_numpy(d_orc.astype(np.float32)).cuda(), torch.from_numpy(d_gpu.astype(np.float32)).cuda(), 0.01, 1.0, 0.1)
    assert ne > 0 and rate >= 0.999
    # back to voxels
    assert eng.set_scoring_grid((1, 1, 1)) == tuple(w["ct"]["n"])
    again = eng.dose(N, seed)
    assert float((again - fine).abs().max()) <= 2e-6 * float(fine.max())
    eng.close()


def test_coarse_influence_columns_against_the_oracle():
    from paper_2307_01416_b200 import binding
    from oracle import vpmc_oracle as O
    w = wl.small_water(n=(24, 24, 40), energy=90.0, sigma=3.0, with_aperture=True, opening_radius=4.0, n_spots=3)
    div = (2, 3, 2)
    hps, thr, seed = 20_000, 1e-3, 6
    eng = binding.Engine(w)
    sn = eng.set_scoring_grid(div)
    mats = eng.influence([binding.scenario(), binding.scenario((2.0, 0.0, 0.0), 0.965)], hps, thr, seed)
    pb = oracle_problem(w)
    for s, sc in enumerate((O.scenario(), O.scenario((2.0, 0.0, 0.0), float(np.float32(0.965))))):
        rp, col, val = (a.cpu().numpy() for a in mats[s])
        assert rp.shape == (eng.n_spots + 1,) and col.max() < eng.ncell
        for g in range(eng.n_spots):
            e, _ = O.influence_edep(pb, g, hps, seed, sc)
            ref = O.dose_from_edep_coarse(pb, e, 1.0 / hps, div).astype(np.float32)
            a = np.zeros(eng.ncell); a[col[rp[g]:rp[g + 1]]] = val[rp[g]:rp[g + 1]]
            assert (np.diff(col[rp[g]:rp[g + 1]]) > 0).all()                       # cell indices ascending, unique
            mx = float(ref.max())
            kept_ref = (ref > 0) & (ref >= np.float32(thr) * ref.max())
            both = (a > 0) & kept_ref
            assert np.abs(a[both] - ref[both]).max() <= 2e-3 * mx                   # re-dealt histories move single deposits
            one = (a > 0) != kept_ref
            assert np.all(np.abs(ref[one] - thr * mx) <= 0.1 * thr * mx + 2e-3 * mx * 0 + 5e-5 * mx), (g, int(one.sum()))
            assert abs(a.sum() - ref[kept_ref].sum()) <= 2e-3 * ref.sum()
    eng.close()
