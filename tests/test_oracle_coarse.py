"""Pins of the oracle's coarse-grid dose (oracle.vpmc_oracle.dose_from_edep_coarse): what the definition
"dose of a cell = its energy / its mass" fixes -- the plain C6 dose for cells of one voxel, the mean of the voxel doses in a
uniform medium, energy conservation in any medium, and smaller cells at a ragged edge."""
import numpy as np

from oracle import vpmc_oracle as orc
from paper_2307_01416_b200 import workloads as wl
from tests.helpers import oracle_problem


def _case(hetero):
    w = wl.small_water(n=(9, 7, 20), h=(2.0, 2.5, 1.5), energy=60.0, sigma=2.0)
    if hetero:
        rng = np.random.default_rng(2)
        w["ct"]["hu"] = rng.integers(-900, 1400, size=w["ct"]["hu"].shape).astype(np.int16)
    return w


def test_cells_of_one_voxel_are_the_plain_dose():
    w = _case(True)
    pb = oracle_problem(w)
    e, _ = orc.dose_edep(pb, 3000, 4)
    a = orc.dose_from_edep_coarse(pb, e, 0.37, (1, 1, 1))
    b = orc.dose_from_edep(pb, e, 0.37)
    assert a.shape == b.shape and np.allclose(a, b, rtol=1e-13, atol=0) and b.max() > 0


def test_uniform_medium_gives_the_mean_of_the_voxel_doses_and_ragged_cells_are_smaller():
    w = _case(False)
    pb = oracle_problem(w)
    e, _ = orc.dose_edep(pb, 3000, 4)
    div = (2, 3, 4)                                    # 9 = 4 x 2 + 1, 7 = 2 x 3 + 1, 20 = 5 x 4: ragged in x and y
    cell, sn = orc.coarse_cells(pb, div)
    assert sn == [5, 3, 5] and cell.max() == 5 * 3 * 5 - 1
    counts = np.bincount(cell)
    assert counts.max() == 24 and counts.min() == 1 * 1 * 4 and counts.sum() == 9 * 7 * 20
    # voxel (8, 6, 19) is alone in x and y in the last cell
    assert cell[8 + 9 * (6 + 7 * 19)] == 4 + 5 * (2 + 3 * 4)
    fine = orc.dose_from_edep(pb, e, 1.0)
    coarse = orc.dose_from_edep_coarse(pb, e, 1.0, div)
    mean = np.bincount(cell, weights=fine) / counts
    assert np.allclose(coarse, mean, rtol=1e-12, atol=0) and coarse.max() > 0


def test_energy_is_conserved_in_any_medium():
    w = _case(True)
    pb = oracle_problem(w)
    e, _ = orc.dose_edep(pb, 3000, 4)
    hu = np.asarray(w["ct"]["hu"], dtype=np.float64).reshape(-1)
    rho = np.maximum(np.array([orc.calib_eval(w["calib"], x)[1] for x in hu]), float(pb.params.rho_min))
    V = 2.0 * 2.5 * 1.5 * 1e-3
    for div in ((2, 2, 2), (3, 1, 5), (9, 7, 20)):
        cell, sn = orc.coarse_cells(pb, div)
        d = orc.dose_from_edep_coarse(pb, e, 1.0, div)
        mass = np.bincount(cell, weights=rho * V, minlength=d.size)
        # sum of dose x mass = deposited energy (MeV -> J/kg g = 1.602e-10)
        assert abs((d * mass).sum() / 1.602176634e-10 - e.sum()) <= 1e-12 * e.sum()
    # one cell for the whole grid: total energy over total mass
    assert d.size == 1 and abs(d[0] - e.sum() / (rho * V).sum() * 1.602176634e-10) <= 1e-12 * d[0]
