"""SURVEY.md 8(f)-2, second half: energy-layer-specific ("dynamic") apertures (the paper's future work).  The
boundary needs no new call for them: a field whose opening changes with the energy layer is handed over as one beam per
layer with the SAME frame, each with its own opening (bitmap or polygon) and that layer's spots.  Checked here against the
oracle given the same beams: dose within 1e-3 of the maximum, gamma 1 %/1 mm >= 99.9 %, tallies, discrete traces (digests)
-- and that the per-layer openings really act: each layer's dose differs from the one-opening plan's."""
import numpy as np
import pytest

from paper_2307_01416_b200 import workloads as wl
from tests.helpers import grid, oracle_problem

pytestmark = pytest.mark.gpu


def layered_case(per_layer=True):
    """Three layers (70, 90, 110 MeV), 5 spots each on a line; openings: a disc of 3 mm, an off-centre polygon slot, a disc of
    6 mm.  per_layer=False: every layer behind the widest opening (the comparison plan)."""
    n, h = (24, 24, 50), (2.0, 2.0, 2.0)
    ct = wl.water_ct(n, h, (-0.5 * n[0] * h[0], -0.5 * n[1] * h[1], 0.0))
    rng = np.random.default_rng(11)
    ct["hu"] = np.rint(rng.normal(20, 30, size=ct["hu"].shape)).astype(np.int16)
    z_iso, face = 30.0, 50.0
    small = wl.aperture(*wl.disc_bitmap(128, 0.1, 3.0), 30.0, face)
    wide = wl.aperture(*wl.disc_bitmap(160, 0.1, 6.0), 30.0, face)
    slot = wl.polygon_aperture([(-1.0, -5.0), (4.0, -5.0), (4.0, 5.0), (-1.0, 5.0)], 30.0, face)
    beams = []
    for energy, ap in ((70.0, small), (90.0, slot), (110.0, wide)):
        sp = [((j - 2) * 2.5, 0.0, energy, 1.0 + 0.25 * j, 3.0) for j in range(5)]
        beams.append(wl.beam(sp, iso=(0, 0, z_iso), aperture=ap if per_layer else wide))
    return {"name": "layered", "ct": ct, "calib": wl.calibration(), "beams": beams}


@pytest.fixture(scope="module")
def bind():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2307_01416_b200 import binding
    binding.lib()
    return binding


def test_one_beam_per_layer_against_the_oracle(bind):
    from oracle import vpmc_oracle as O
    w = layered_case()
    N, seed = 150_000, 9
    eng = bind.Engine(w)
    pb = oracle_problem(w)
    d_gpu = eng.dose(N, seed).cpu().numpy().astype(np.float64)
    tg = eng.tallies().as_dict()
    d_orc, to = O.dose(pb, N, seed)
    to = to.as_dict()
    assert np.isfinite(d_gpu).all()
    err = np.abs(d_gpu - d_orc).max() / d_orc.max()
    gam = O.gamma_pass_rate(grid(w, d_orc), grid(w, d_gpu), w["ct"]["h"], dd=0.01, dta=1.0, thr=0.1)
    n_dig = 20000
    a = eng.digests(N, seed, 0, n_dig)
    b = O.digests(pb, N, seed, 0, n_dig)
    differ = (a["hash"] != b["hash"]) | (a["n_rec"] != b["n_rec"])
    print("layer apertures: max |dD|/Dmax = %.3e gamma %.5f, %d of %d traces differ" % (err, gam, differ.sum(), n_dig))
    assert err < 1e-3 and gam >= 0.999
    assert differ.sum() <= 1e-3 * n_dig
    cnt = ("n_stopped_ct", "n_stopped_rs", "n_stopped_brass", "n_nuclear", "n_escaped")
    assert sum(tg[k] for k in cnt) == N
    for k in cnt:
        assert abs(int(tg[k]) - int(to[k])) <= max(2, 1e-3 * N), (k, tg[k], to[k])
    eng.close()


def test_the_layers_see_their_own_openings(bind):
    """Against the plan with the widest opening on every layer: more protons end in the brass, and the dose of the layers
    behind the narrow openings (the proximal part of the depth-dose) drops while the last layer's peak region keeps its dose."""
    N, seed = 150_000, 9
    e1, e0 = bind.Engine(layered_case(True)), bind.Engine(layered_case(False))
    d1, d0 = e1.dose(N, seed).cpu().numpy().astype(np.float64), e0.dose(N, seed).cpu().numpy().astype(np.float64)
    t1, t0 = e1.tallies().as_dict(), e0.tallies().as_dict()
    assert t1["n_stopped_brass"] > 1.2 * t0["n_stopped_brass"]
    n = (24, 24, 50)
    z1, z0 = d1.reshape(n[2], n[1], n[0]).sum(axis=(1, 2)), d0.reshape(n[2], n[1], n[0]).sum(axis=(1, 2))
    k70 = int(np.argmax(z0[:25]))                      # Bragg peak of the 70 MeV layer (~41 mm deep)
    assert z1[k70] < 0.9 * z0[k70]
    k110 = 40 + int(np.argmax(z0[40:]))                # of the 110 MeV layer (~90 mm): same opening in both plans
    assert abs(z1[k110] - z0[k110]) <= 0.05 * z0[k110]
    e1.close(); e0.close()
