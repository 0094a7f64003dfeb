"""Pins of the oracle's polygon opening ("the opening boundary ... crossing number", ref. 67):
the point test against an independent algorithm (winding angle) and closed shapes, a rectangle on the pixel grid against the
already pinned bitmap path (history by history), and the pass fraction against the Gaussian mass over the opening."""
import math

import numpy as np

from oracle import vpmc_oracle as orc
from paper_2307_01416_b200 import workloads as wl
from tests.helpers import oracle_problem


def _winding_inside(poly, x, y):
    """Sum of the signed angles subtended by the edges at (x, y): +-2 pi inside, 0 outside (another algorithm than the oracle's)."""
    p = np.asarray(poly, dtype=np.float64) - np.array([x, y])
    q = np.roll(p, -1, axis=0)
    ang = np.arctan2(p[:, 0] * q[:, 1] - p[:, 1] * q[:, 0], (p * q).sum(axis=1)).sum()
    return abs(ang) > math.pi


def test_point_in_polygon_against_closed_shapes_and_the_winding_angle():
    square = [(-1, -2), (3, -2), (3, 2), (-1, 2)]
    assert orc.point_in_polygon(square, 0, 0) and orc.point_in_polygon(square, 2.9, -1.9)
    assert not orc.point_in_polygon(square, 3.1, 0) and not orc.point_in_polygon(square, 0, 2.1) and not orc.point_in_polygon(square, -1.1, 0)
    # concave "L": the notch is outside
    ell = [(0, 0), (4, 0), (4, 1), (1, 1), (1, 4), (0, 4)]
    assert orc.point_in_polygon(ell, 0.5, 3.0) and orc.point_in_polygon(ell, 3.0, 0.5) and not orc.point_in_polygon(ell, 2.0, 2.0)
    # vertex order does not matter
    assert orc.point_in_polygon(ell[::-1], 0.5, 3.0) and not orc.point_in_polygon(ell[::-1], 2.0, 2.0)
    # the star of config 5 on random points, against the winding angle
    star = wl.config5(polygon=True)["beams"][0]["aperture"]["polygon"]
    rng = np.random.default_rng(4)
    pts = rng.uniform(-22, 22, size=(4000, 2))
    got = np.array([orc.point_in_polygon(star, x, y) for x, y in pts])
    ref = np.array([_winding_inside(star, x, y) for x, y in pts])
    assert np.array_equal(got, ref) and 0.2 < got.mean() < 0.6
    # and the bitmap of the same star is this test at the pixel centres (workloads.polygon_bitmap): sampled pixels
    op, u0, v0, du, dv = wl.polygon_bitmap(1024, 0.1, star)
    for iy, ix in rng.integers(300, 724, size=(500, 2)):
        assert bool(op[iy, ix]) == orc.point_in_polygon(star, float(u0) + (ix + 0.5) * float(du), float(v0) + (iy + 0.5) * float(dv))


def _slot_case(polygon):
    """One 100 MeV spot through an off-centre 2 x 6 mm slot (asymmetric in x and y), edges on the 0.1 mm pixel grid."""
    w = wl.small_water(n=(20, 20, 40), energy=100.0, sigma=3.0, with_aperture=True)
    x0, x1, y0, y1 = 0.5, 2.5, -4.0, 2.0
    if polygon:
        w["beams"][0]["aperture"] = wl.polygon_aperture([(x0, y0), (x1, y0), (x1, y1), (x0, y1)], 30.0, 40.0)
    else:
        n = 128
        u0 = -6.4
        c = u0 + (np.arange(n) + 0.5) * 0.1
        X, Y = np.meshgrid(c, c, indexing="xy")
        op = ((X > x0) & (X < x1) & (Y > y0) & (Y < y1)).astype(np.uint8)
        w["beams"][0]["aperture"] = wl.aperture(op, u0, u0, 0.1, 0.1, 30.0, 40.0)
    return w, (x0, x1, y0, y1)


def test_rectangle_polygon_equals_the_bitmap_path_history_by_history():
    """The same opening given as a polygon and as a bitmap whose pixel edges are the polygon's edges: every history takes the
    same steps (a position exactly on an edge has probability zero), so dose, tallies and digests are identical."""
    wp, _ = _slot_case(True)
    wb, _ = _slot_case(False)
    N, seed = 6000, 21
    dp, tp = orc.dose(oracle_problem(wp), N, seed)
    db, tb = orc.dose(oracle_problem(wb), N, seed)
    assert tp.as_dict() == tb.as_dict()
    assert np.array_equal(dp, db) and dp.sum() > 0
    gp = orc.digests(oracle_problem(wp), N, seed, 0, 500)
    gb = orc.digests(oracle_problem(wb), N, seed, 0, 500)
    assert np.array_equal(gp["hash"], gb["hash"]) and np.array_equal(gp["n_rec"], gb["n_rec"])
    # transposing the slot (x <-> y) is a different opening: the polygon's axes are not swapped anywhere
    wt, (x0, x1, y0, y1) = _slot_case(True)
    wt["beams"][0]["aperture"] = wl.polygon_aperture([(y0, x0), (y1, x0), (y1, x1), (y0, x1)], 30.0, 40.0)
    dt, _ = orc.dose(oracle_problem(wt), N, seed)
    assert not np.array_equal(dt, dp)


def test_pass_fraction_is_the_gaussian_mass_over_the_polygon():
    """Scattering off: a history reaches the CT iff its (unchanged) lateral position lies in the opening; brass stops 100 MeV
    (P:L81).  Number reaching the CT = N x Gaussian mass over the slot (product of erf differences), within 4 sigma."""
    w, (x0, x1, y0, y1) = _slot_case(True)
    p = orc.default_params(flags=0)
    N = 20000
    _, tal = orc.dose(oracle_problem(w, params=p), N, 3)
    sig = 3.0
    phi = lambda z: 0.5 * (1.0 + math.erf(z / (sig * math.sqrt(2.0))))
    mass = (phi(x1) - phi(x0)) * (phi(y1) - phi(y0))
    n_ct = tal.n_stopped_ct + tal.n_escaped
    assert tal.n_stopped_brass == N - n_ct
    assert abs(n_ct - N * mass) < 4.0 * math.sqrt(N * mass * (1 - mass)), (n_ct, N * mass)
