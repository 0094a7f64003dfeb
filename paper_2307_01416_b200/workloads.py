"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json configs).

This module serves BOTH the CPU oracle (tests) and the CUDA path (tests, bench).  It holds none of the
method's arithmetic: it only lays out CT grids, calibration nodes, spot lattices and opening bitmaps as
plain numpy arrays.  Every real number it emits is an exact fp32 value, so the fp64 oracle and the fp32
kernels start from identical inputs.  (The only physics-flavoured lines are in the *plan design* of the
head cases -- picking energy layers that reach a target -- which is an input choice, not transport.)

Problem format (dict):
  ct     = {n: (nx,ny,nz), h: (hx,hy,hz) mm, origin: low corner of voxel (0,0,0) mm, hu: int16 [nz,ny,nx]}
  calib  = {hu, rsp, rho: fp32 node arrays ascending in hu, xsp: None}
  beams  = [{iso: (3,), rot: (3,3) with r_ct = iso + rot @ r_beam, spots: fp32 [n,5] = x, y, E, weight, sigma,
             rs_wet: mm (0 = none), rs_face: mm upstream of isocentre, aperture: None or
             {T, face, open: uint8 [ny,nx], u0, v0, du, dv}}]
"""
from __future__ import annotations

import numpy as np

F = np.float32

# synthetic piecewise-linear calibration: (HU, RSP, rho)
CALIB_NODES = np.array([(-1000, 0.001, 0.0012), (0, 1.0, 1.0), (100, 1.08, 1.09),
                        (1000, 1.55, 1.60), (3000, 2.5, 2.8)], dtype=np.float64)


def calibration():
    return {"hu": CALIB_NODES[:, 0].astype(F), "rsp": CALIB_NODES[:, 1].astype(F),
            "rho": CALIB_NODES[:, 2].astype(F), "xsp": None}


def spot_sigma(E):
    """In-air spot sigma, linear 5 mm @ 71.3 MeV -> 2 mm @ 228.8 MeV."""
    E = np.asarray(E, dtype=np.float64)
    return (5.0 + (E - 71.3) * (2.0 - 5.0) / (228.8 - 71.3)).astype(F)


def disc_bitmap(n_pix: int, pitch: float, radius: float, centre=(0.0, 0.0)):
    """Opening bitmap: pixel (iy, ix) open iff its centre lies within `radius` of `centre` (beam frame, mm).
    Returns (open uint8 [n,n], u0, v0, du, dv) with the bitmap centred on (0, 0)."""
    u0 = v0 = -0.5 * n_pix * pitch
    c = u0 + (np.arange(n_pix, dtype=np.float64) + 0.5) * pitch
    X, Y = np.meshgrid(c, c, indexing="xy")
    op = ((X - centre[0]) ** 2 + (Y - centre[1]) ** 2 <= radius ** 2).astype(np.uint8)
    return op, F(u0), F(v0), F(pitch), F(pitch)


def polygon_bitmap(n_pix: int, pitch: float, poly_xy: np.ndarray):
    """Rasterise a closed polygon by the crossing-number test at pixel centres (ref 67)."""
    u0 = v0 = -0.5 * n_pix * pitch
    c = u0 + (np.arange(n_pix, dtype=np.float64) + 0.5) * pitch
    X, Y = np.meshgrid(c, c, indexing="xy")
    inside = np.zeros(X.shape, dtype=bool)
    P = np.asarray(poly_xy, dtype=np.float64)
    for k in range(len(P)):
        x1, y1 = P[k]
        x2, y2 = P[(k + 1) % len(P)]
        if y1 == y2:
            continue
        cond = (y1 > Y) != (y2 > Y)
        xi = x1 + (Y - y1) * (x2 - x1) / (y2 - y1)
        inside ^= cond & (X < xi)
    return inside.astype(np.uint8), F(u0), F(v0), F(pitch), F(pitch)


def water_ct(n, h, origin):
    return {"n": tuple(int(x) for x in n), "h": tuple(F(x) for x in h), "origin": tuple(F(x) for x in origin),
            "hu": np.zeros((n[2], n[1], n[0]), dtype=np.int16)}


def beam(spots, iso, rot=None, rs_wet=0.0, rs_face=190.0, aperture=None):
    return {"iso": np.asarray(iso, dtype=F), "rot": np.eye(3, dtype=F) if rot is None else np.asarray(rot, dtype=F),
            "spots": np.asarray(spots, dtype=F).reshape(-1, 5), "rs_wet": F(rs_wet), "rs_face": F(rs_face),
            "aperture": aperture}


def aperture(open_u8, u0, v0, du, dv, T=30.0, face=150.0):
    return {"T": F(T), "face": F(face), "open": np.ascontiguousarray(open_u8, dtype=np.uint8),
            "u0": F(u0), "v0": F(v0), "du": F(du), "dv": F(dv)}


# ------------------------------------------------------------------------------------------ configs

def config1(n_histories: int = 100_000, seed: int = 1):
    """BASELINE.json configs[0]: water 50x50x100 @ 2 mm, one 100 MeV spot sigma 4 mm on axis, 30 mm brass,
    2 cm circular opening, downstream face 100 mm upstream of the surface, no range shifter."""
    ct = water_ct((50, 50, 100), (2, 2, 2), (-50, -50, 0))
    op, u0, v0, du, dv = disc_bitmap(512, 0.1, 10.0)
    z_iso = 50.0   # isocentre 50 mm deep -> block face 150 mm upstream of it = 100 mm upstream of the surface
    b = beam([[0, 0, 100, 1, 4]], iso=(0, 0, z_iso), aperture=aperture(op, u0, v0, du, dv, 30.0, z_iso + 100.0))
    return {"name": "config1", "ct": ct, "calib": calibration(), "beams": [b], "n_histories": n_histories, "seed": seed}


def config2_plans():
    return [(d, rs) for rs in (False, True) for d in (10, 20, 30, 40)]


def config2(opening_mm: int = 20, range_shifter: bool = False, n_histories: int = 10_000_000, seed: int = 2):
    """BASELINE.json configs[1]: water 100x100x150 @ 2 mm; 30 mm brass, circular opening 1/2/3/4 cm, with or without a
    45 mm WET range shifter; 5 mm spot lattice over opening + 5 mm margin; 33 layers 70..150 MeV; uniform weights."""
    ct = water_ct((100, 100, 150), (2, 2, 2), (-100, -100, 0))
    op, u0, v0, du, dv = disc_bitmap(512, 0.1, 0.5 * opening_mm)
    half = 0.5 * opening_mm + 5.0
    k = int(np.floor(half / 5.0 + 1e-9))
    xs = np.arange(-k, k + 1, dtype=np.float64) * 5.0
    energies = 70.0 + 2.5 * np.arange(33)
    spots = [(x, y, E, 1.0, float(spot_sigma(E))) for E in energies for y in xs for x in xs]
    b = beam(spots, iso=(0, 0, 100.0), rs_wet=45.0 if range_shifter else 0.0, rs_face=190.0,
             aperture=aperture(op, u0, v0, du, dv, 30.0, 150.0))
    return {"name": "config2_d%d_%s" % (opening_mm, "rs" if range_shifter else "nors"), "ct": ct,
            "calib": calibration(), "beams": [b], "n_histories": n_histories, "seed": seed}


def small_water(n=(8, 8, 40), h=(2.0, 2.0, 2.0), energy=70.0, sigma=1.5, with_aperture=False, rs_wet=0.0,
                opening_radius=3.0, n_spots=1, z_iso=20.0):
    """Small homogeneous cases for unit tests."""
    ct = water_ct(n, h, (-0.5 * n[0] * h[0], -0.5 * n[1] * h[1], 0.0))
    ap = None
    if with_aperture:
        op, u0, v0, du, dv = disc_bitmap(128, 0.1, opening_radius)
        ap = aperture(op, u0, v0, du, dv, 30.0, z_iso + 20.0)
    rs_face = z_iso + 60.0
    sp = [((j - 0.5 * (n_spots - 1)) * 2.0, 0.0, energy, 1.0 + j, sigma) for j in range(n_spots)]
    return {"name": "small_water", "ct": ct, "calib": calibration(),
            "beams": [beam(sp, iso=(0, 0, z_iso), rs_wet=rs_wet, rs_face=rs_face, aperture=ap)]}
