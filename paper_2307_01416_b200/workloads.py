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
             {T, face, open: uint8 [ny,nx], u0, v0, du, dv} (opening bitmap) or
             {T, face, polygon: fp32 [n,2]} (the opening's boundary polygon, tested on the device: SURVEY.md 8(f)-2)}]
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


def polygon_aperture(poly_xy, T=30.0, face=150.0):
    """Aperture whose opening is the closed polygon poly_xy [n, 2] (beam frame, mm), exact fp32 vertices."""
    return {"T": F(T), "face": F(face), "polygon": np.ascontiguousarray(np.asarray(poly_xy, dtype=F).reshape(-1, 2))}


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


# ------------------------------------------------------------------------------------------ configs 3-5
# Plan design below (which energies reach the target, whether a range shifter is needed) uses the water-equivalent
# depth along the beam axis.  It is an INPUT choice made by the harness, like a planning system's; no transport code.

ALPHA, P_EXP = 0.022, 1.77


def _rsp_of_hu(hu):
    return np.interp(hu, CALIB_NODES[:, 0], CALIB_NODES[:, 1])


def _range_w(E):
    return ALPHA * np.asarray(E, dtype=np.float64) ** P_EXP


def _energy_of_range(R):
    return (np.asarray(R, dtype=np.float64) / ALPHA) ** (1.0 / P_EXP)


def _beam_rot(direction):
    """rot (3x3, columns = beam axes in the CT frame) with the third column = direction of travel."""
    w = np.asarray(direction, dtype=np.float64)
    w = w / np.linalg.norm(w)
    a = np.array([0.0, 0.0, 1.0]) if abs(w[2]) < 0.9 else np.array([1.0, 0.0, 0.0])
    u = np.cross(a, w); u /= np.linalg.norm(u)
    v = np.cross(w, u)
    return np.stack([u, v, w], axis=1).astype(F)


def _wet_profile(ct, iso, direction, s_lo, s_hi, ds=0.5):
    """water-equivalent path length along iso + s*direction for s in [s_lo, s_hi], starting at 0 at s_lo."""
    n, h, o = np.array(ct["n"]), np.array(ct["h"], dtype=np.float64), np.array(ct["origin"], dtype=np.float64)
    s = np.arange(s_lo, s_hi, ds) + 0.5 * ds
    p = np.asarray(iso, dtype=np.float64)[None, :] + s[:, None] * np.asarray(direction, dtype=np.float64)[None, :]
    idx = np.floor((p - o) / h).astype(np.int64)
    inside = ((idx >= 0) & (idx < n)).all(axis=1)
    idx = np.clip(idx, 0, n - 1)
    hu = ct["hu"][idx[:, 2], idx[:, 1], idx[:, 0]].astype(np.float64)
    rsp = np.where(inside, _rsp_of_hu(hu), 0.0)
    return s + 0.5 * ds, np.cumsum(rsp * ds)


def _ct_min_w(ct, iso, rot):
    n, h, o = np.array(ct["n"]), np.array(ct["h"], dtype=np.float64), np.array(ct["origin"], dtype=np.float64)
    lo, hi = o, o + n * h
    w = np.asarray(rot, dtype=np.float64)[:, 2]
    return min(float(np.dot(np.where([(k >> a) & 1 for a in range(3)], hi, lo) - np.asarray(iso, dtype=np.float64), w)) for k in range(8))


def head_ct(seed: int = 3):
    """Synthetic head: 256x256x160 voxels of 1x1x1.5 mm, ellipsoid skull shell +1000 HU,
    brain N(40, 20^2) HU, three air cavities, outside air."""
    rng = np.random.default_rng(seed)
    n, h = (256, 256, 160), (1.0, 1.0, 1.5)
    origin = (-128.0, -128.0, -120.0)
    x = origin[0] + (np.arange(n[0]) + 0.5) * h[0]
    y = origin[1] + (np.arange(n[1]) + 0.5) * h[1]
    z = origin[2] + (np.arange(n[2]) + 0.5) * h[2]
    Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
    ax_o = np.array([80.0, 100.0, 105.0]); ax_i = ax_o - 7.0
    e_o = (X / ax_o[0]) ** 2 + (Y / ax_o[1]) ** 2 + (Z / ax_o[2]) ** 2
    e_i = (X / ax_i[0]) ** 2 + (Y / ax_i[1]) ** 2 + (Z / ax_i[2]) ** 2
    hu = np.full(X.shape, -1000.0)
    hu[e_o <= 1.0] = 1000.0
    brain = e_i <= 1.0
    hu[brain] = np.rint(rng.normal(40.0, 20.0, size=int(brain.sum())))
    for _ in range(3):                                    # air cavities, lower-anterior interior
        r = rng.uniform(8.0, 15.0)
        c = np.array([rng.uniform(-25, 25), rng.uniform(35, 60), rng.uniform(-70, -35)])
        hu[((X - c[0]) ** 2 + (Y - c[1]) ** 2 + (Z - c[2]) ** 2 <= r * r) & brain] = -1000.0
    return {"n": n, "h": tuple(F(v) for v in h), "origin": tuple(F(v) for v in origin), "hu": hu.astype(np.int16)}


def _plan_beam(ct, target_c, r_t, direction, pitch, layer_step=2.5, margin_spots=5.0, margin_ap=3.0, bitmap_pitch=0.1):
    """One beam on a spherical target: isocentre = target centre; aperture opening = BEV projection + margin_ap;
    spot lattice within r_t + margin_spots; layers every layer_step MeV over the target's WET extent +- one layer;
    range shifter iff the proximal edge is shallower than R_w(71.3 MeV) + 5 mm (Table 1 of the paper: "Range Shifter
    Yes/No")."""
    rot = _beam_rot(direction)
    d = rot[:, 2].astype(np.float64)
    wmin = _ct_min_w(ct, target_c, rot)
    s, wet = _wet_profile(ct, target_c, d, wmin, r_t + 1.0)
    wet_prox = float(np.interp(-r_t, s, wet)); wet_dist = float(np.interp(r_t, s, wet))
    use_rs = wet_prox < float(_range_w(71.3)) + 5.0
    extra = 45.0 if use_rs else 0.0
    e_lo = float(_energy_of_range(wet_prox + extra)) - layer_step
    e_hi = float(_energy_of_range(wet_dist + extra)) + layer_step
    energies = np.arange(np.ceil(max(e_lo, 70.0) / layer_step) * layer_step, min(e_hi, 230.0) + 1e-9, layer_step)
    k = int(np.floor((r_t + margin_spots) / pitch + 1e-9))
    g = np.arange(-k, k + 1) * pitch
    lat = [(x, y) for y in g for x in g if x * x + y * y <= (r_t + margin_spots) ** 2 + 1e-9]
    spots = [(x, y, E, 1.0, float(spot_sigma(E))) for E in energies for (x, y) in lat]
    n_pix = int(2 ** np.ceil(np.log2(2.0 * (r_t + margin_ap + 2.0) / bitmap_pitch)))
    op, u0, v0, du, dv = disc_bitmap(n_pix, bitmap_pitch, r_t + margin_ap)
    # devices ride 150 / 190 mm upstream of the isocentre unless the CT box (with its air) reaches further
    face = max(150.0, np.ceil(-wmin) + 5.0)
    return beam(spots, iso=target_c, rot=rot, rs_wet=45.0 if use_rs else 0.0, rs_face=face + 40.0,
                aperture=aperture(op, u0, v0, du, dv, 30.0, face))


def config3(seed: int = 3, n_histories: int = 10_000_000, pitch: float = 2.5):
    """BASELINE.json configs[2]: head CT, spherical target of volume log-uniform in 0.4-43 cc, 2 beams (the second
    rotated 60 degrees about z), apertures = target projection + 3 mm, 2.5 mm spot pitch."""
    ct = head_ct(seed)
    rng = np.random.default_rng(seed + 1000)
    vol = np.exp(rng.uniform(np.log(0.4), np.log(43.0)))              # cc
    r_t = float((3.0 * vol * 1000.0 / (4.0 * np.pi)) ** (1.0 / 3.0))  # mm
    phi = rng.uniform(-0.35, 0.35) + (np.pi if rng.random() < 0.5 else 0.0)      # lateral, tilted <= 20 degrees
    d_t = np.array([np.cos(phi), np.sin(phi), rng.uniform(-0.2, 0.2)]); d_t /= np.linalg.norm(d_t)
    ax_i = np.array([73.0, 93.0, 98.0])
    t_surf = 1.0 / np.sqrt(((d_t / ax_i) ** 2).sum())                 # inner skull surface along d_t
    depth = rng.uniform(15.0, 40.0) + r_t
    c = np.round(d_t * max(t_surf - depth, 0.0), 1).astype(np.float64)
    dir1 = -d_t                                                       # shallowest approach
    ca, sa = np.cos(np.pi / 3), np.sin(np.pi / 3)
    dir2 = np.array([ca * dir1[0] - sa * dir1[1], sa * dir1[0] + ca * dir1[1], dir1[2]])
    beams = [_plan_beam(ct, c, r_t, dir1, pitch), _plan_beam(ct, c, r_t, dir2, pitch)]
    return {"name": "config3_seed%d" % seed, "ct": ct, "calib": calibration(), "beams": beams, "n_histories": n_histories,
            "seed": seed, "target": {"centre": c, "radius": r_t, "volume_cc": float(vol)}}


SCENARIOS13 = ([((0.0, 0.0, 0.0), 1.0)] +
               [(tuple(float(s) * 3.0 if a == k else 0.0 for a in range(3)), 1.0) for k in range(3) for s in (+1, -1)] +
               [((0.0, 0.0, 0.0), 1.035), ((0.0, 0.0, 0.0), 0.965)] +
               [((0.0, 0.0, float(sz) * 3.0), sc) for sc in (1.035, 0.965) for sz in (+1, -1)])


def config4(hist_per_spot: int = 10_000, lo: int = 1800, hi: int = 2200, max_seed: int = 64):
    """BASELINE.json configs[3]: influence-matrix build on a config-3 head with about 2000 spots (the first seed whose
    plan has lo..hi spots over its 2 beams), 13 scenarios (SCENARIOS13: 3 mm, 3.5 %), threshold 1e-4."""
    for seed in range(3, 3 + max_seed):
        rng = np.random.default_rng(seed + 1000)
        vol = np.exp(rng.uniform(np.log(0.4), np.log(43.0)))
        if not (3.0 < vol < 14.0):                         # cheap pre-filter: spot count grows with the target volume
            continue
        w = config3(seed)
        n = sum(b["spots"].shape[0] for b in w["beams"])
        if lo <= n <= hi:
            w["name"] = "config4_seed%d" % seed
            w["hist_per_spot"] = hist_per_spot
            w["scenarios"] = SCENARIOS13
            w["rel_threshold"] = 1e-4
            return w
    raise RuntimeError("no seed gives %d..%d spots" % (lo, hi))


def star_polygon(a, ph, n_vertices: int = 720):
    """Config 5's irregular opening: r(phi) = 15 mm (1 + sum_{k=2..6} a_k cos(k phi + phi_k)); fp32 vertices."""
    phi = np.linspace(0.0, 2 * np.pi, n_vertices, endpoint=False)
    r = 15.0 * (1.0 + sum(a[i] * np.cos((i + 2) * phi + ph[i]) for i in range(5)))
    return np.stack([r * np.cos(phi), r * np.sin(phi)], axis=1).astype(F)


def config5(seed: int = 5, n_histories: int = 100_000_000, polygon: bool = False):
    """BASELINE.json configs[4]: 512x512x200 voxels of 1 mm, random z-slabs (-1000..+1500 HU), 45 mm WET range shifter,
    30 mm brass with a star-shaped opening (bitmap 1024^2 @ 0.1 mm), 65 layers 70..230 MeV, 5 mm lattice.
    polygon=True: the same opening handed over as its boundary polygon instead of the rasterised bitmap."""
    rng = np.random.default_rng(seed)
    n, h = (512, 512, 200), (1.0, 1.0, 1.0)
    hu = np.empty((n[2], n[1], n[0]), dtype=np.int16)
    z = 0
    while z < n[2]:
        t = int(rng.integers(4, 33))
        hu[z:z + t] = np.int16(rng.integers(-1000, 1501))
        z += t
    ct = {"n": n, "h": tuple(F(v) for v in h), "origin": (F(-256.0), F(-256.0), F(0.0)), "hu": hu}
    poly = star_polygon(rng.uniform(0.0, 0.12, size=5), rng.uniform(0.0, 2 * np.pi, size=5))      # a_k in U[0, 0.12]
    if polygon:
        ap = polygon_aperture(poly, 30.0, 150.0)
    else:
        op, u0, v0, du, dv = polygon_bitmap(1024, 0.1, poly)
        ap = aperture(op, u0, v0, du, dv, 30.0, 150.0)
    half = np.ceil(np.abs(poly.astype(np.float64)).max() / 5.0) * 5.0 + 5.0
    g = np.arange(-half, half + 1e-9, 5.0)
    energies = 70.0 + 2.5 * np.arange(65)
    spots = [(x, y, E, 1.0, float(spot_sigma(E))) for E in energies for y in g for x in g]
    b = beam(spots, iso=(0.0, 0.0, 100.0), rs_wet=45.0, rs_face=190.0, aperture=ap)
    return {"name": "config5" + ("_polygon" if polygon else ""), "ct": ct, "calib": calibration(), "beams": [b], "n_histories": n_histories, "seed": seed}
