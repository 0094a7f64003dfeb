"""The on-GPU stopping rule (SURVEY.md 8(d) metric 2, 8(f)-3; "<0.5 %") against the oracle's plain loop
(oracle.vpmc_oracle.dose_to_uncertainty): batches of N_b histories with ids k 2^32 + i, the C6 estimator after each,
stop at the first batch count >= min_batches whose estimate is <= target.  The decision is an integer taken from a
floating-point estimate, so the test picks its target halfway (geometrically) between two consecutive estimates of the
oracle's sequence: both sides must then stop after the same number of batches."""
import math

import numpy as np
import pytest

from paper_2307_01416_b200 import workloads as wl
from tests.helpers import oracle_problem

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def bind():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2307_01416_b200 import binding
    binding.lib()
    return binding


def case():
    return wl.small_water(n=(20, 20, 40), energy=80.0, sigma=3.0, n_spots=3, with_aperture=True, opening_radius=6.0)


def test_stops_after_the_same_batch_as_the_oracle_loop(bind):
    from oracle import vpmc_oracle as O
    w = case()
    pb = oracle_problem(w)
    nb, seed = 20000, 11
    _, _, hist = O.dose_to_uncertainty(pb, nb, 0.0, seed, max_batches=9)        # target 0: the whole sequence of estimates
    assert len(hist) == 8 and all(a > 0 for a in hist)
    # hist[i] = estimate after i + 2 batches.  Target between two consecutive estimates, no estimate within 2 % of it
    target = None
    for k in range(len(hist) - 1, 1, -1):
        t = math.sqrt(hist[k] * hist[k - 1])
        if hist[k] < hist[k - 1] and min(abs(math.log(x / t)) for x in hist) > 0.02:
            target = t
            break
    assert target is not None
    d_orc, n_orc, _ = O.dose_to_uncertainty(pb, nb, target, seed, max_batches=9)
    assert n_orc == next(i + 2 for i, x in enumerate(hist) if x <= target)
    eng = bind.Engine(w)
    d = eng.dose_to_uncertainty(nb, target, seed, max_batches=9).cpu().numpy().astype(np.float64)
    n_gpu, unc, reached = eng.run_info()
    t = eng.tallies().as_dict()
    print("stopping rule: oracle", n_orc, "batches, estimates", ["%.5f" % x for x in hist], "| gpu", n_gpu, "batches, estimate %.5f" % unc, "target %.5f" % target)
    assert n_gpu == n_orc and reached
    assert abs(unc - hist[n_orc - 2]) <= 0.02 * hist[n_orc - 2]
    assert np.isfinite(d).all()
    assert np.abs(d - d_orc).max() <= 1e-3 * d_orc.max()
    assert sum(t[c] for c in ("n_stopped_ct", "n_stopped_rs", "n_stopped_brass", "n_nuclear", "n_escaped")) == n_gpu * nb
    eng.close()


def test_batch_ids_min_and_max_batches(bind):
    from oracle import vpmc_oracle as O
    w = case()
    pb = oracle_problem(w)
    nb, seed = 30000, 12
    eng = bind.Engine(w)
    # target 0 is never reached: max_batches stops the loop
    d3 = eng.dose_to_uncertainty(nb, 0.0, seed, max_batches=3).cpu().numpy().astype(np.float64)
    assert eng.run_info()[0] == 3 and not eng.run_info()[2]
    e = np.zeros(pb.nvox)
    for k in range(3):
        O.dose_edep(pb, nb, seed, hid_offset=k << 32, edep=e)           # D:R15: batch k = ids k 2^32 + i
    d_orc = O.dose_from_edep(pb, e, pb.total_weight / (3 * nb))
    assert np.abs(d3 - d_orc).max() <= 1e-3 * d_orc.max()
    # a huge target is reached at once, but never before min_batches (and never before 2)
    eng.dose_to_uncertainty(nb, 1.0, seed, min_batches=4, max_batches=9)
    assert eng.run_info()[0] == 4 and eng.run_info()[2]
    eng.dose_to_uncertainty(nb, 1.0, seed, min_batches=0, max_batches=9)
    assert eng.run_info()[0] == 2
    # one batch only: no estimate
    d1 = eng.dose_to_uncertainty(nb, 1.0, seed, max_batches=1).cpu().numpy()
    b, u, r = eng.run_info()
    assert b == 1 and u == 0.0 and not r
    # the first batch is the plain dose run of the same ids (high word 0)
    d_plain = eng.dose(nb, seed).cpu().numpy()
    assert np.abs(d1 - d_plain).max() <= 1e-5 * d_plain.max()      # fp32 sums in another order (10 batch grids vs one)
    with pytest.raises(bind.VpmcError):
        eng.dose_to_uncertainty(1 << 24, 0.01, seed)        # larger than the chunk
    eng.close()
