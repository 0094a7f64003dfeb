"""Pins of the CPU oracle against what the paper and the physics fix.

Nothing here compares the oracle with itself or with the CUDA path: expectations are the cited golden
values under tests/golden/, closed forms evaluated in the test, invariants, or an independent numerical
integration (Fermi-Eyges, Bohr).
"""
import math

import numpy as np
import pytest

from oracle import vpmc_oracle as orc
from paper_2307_01416_b200 import workloads as wl
from tests.helpers import oracle_problem, read_golden, grid

ALPHA, P = 0.022, 1.77
MP = 938.272


def golden(kind):
    return [(float(r[1]), float(r[2])) for r in read_golden("physics_pins.txt") if r[0] == kind]


def pencil_water(energy, nz, hz=1.0, sigma=0.0, nxy=5, hxy=400.0, **kw):
    """One pencil spot on the axis of a water column wide enough that nothing leaves sideways."""
    w = wl.small_water(n=(nxy, nxy, nz), h=(hxy, hxy, hz), energy=energy, sigma=sigma, **kw)
    return w


def flags(**on):
    f = 0
    if on.get("mcs"): f |= orc.FLAG_MCS
    if on.get("straggle"): f |= orc.FLAG_STRAGGLE
    if on.get("nuclear"): f |= orc.FLAG_NUCLEAR
    return f


# ------------------------------------------------------------------------------------------ P1

def test_philox_known_answers():
    rows = read_golden("philox_kat.txt")
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        assert orc.philox4x32_10(v[0:4], v[4:6]) == v[6:10]


def test_philox_counter_and_key_sensitivity():
    # every counter word and key word must matter (a dropped word would collide)
    base = orc.philox4x32_10([1, 2, 3, 4], [5, 6])
    for i in range(4):
        c = [1, 2, 3, 4]; c[i] ^= 1
        assert orc.philox4x32_10(c, [5, 6]) != base
    for i in range(2):
        k = [5, 6]; k[i] ^= 1
        assert orc.philox4x32_10([1, 2, 3, 4], k) != base


def test_u01_is_fp32_exact_and_open():
    for x in (0, 1, 511, 512, 0x7FFFFFFF, 0xFFFFFFFF, 0x12345678):
        u = orc.u01(x)
        assert 0.0 < u < 1.0
        assert float(np.float32(u)) == u
        assert u == (2 * (x >> 9) + 1) / 2.0 ** 24
    assert orc.u01(0) == 2.0 ** -24 and orc.u01(0xFFFFFFFF) == 1.0 - 2.0 ** -24


def test_uniform_moments():
    xs = np.array([orc.u01(orc.philox4x32_10([i, 0, 0, 0], [7, 0])[k]) for i in range(4000) for k in range(4)])
    assert abs(xs.mean() - 0.5) < 4 * (1 / math.sqrt(12 * xs.size))
    assert abs(xs.var() - 1 / 12) < 0.004


# ------------------------------------------------------------------------------------------ P2

@pytest.mark.parametrize("E,R0", golden("range_mm"))
def test_csda_range_in_water(E, R0):
    """Loss only: the history stops within R_cut upstream of alpha E^p, for any voxel size."""
    assert abs(ALPHA * E ** P - R0) < 5e-4 * R0
    for hz in (1.0, 2.0, 3.7):
        nz = int(R0 / hz) + 4
        w = pencil_water(E, nz, hz)
        pb = oracle_problem(w, orc.default_params(flags=0))
        rec = orc.trace(pb, [0], 1, 1)[0]
        assert rec[-1]["cause"] == orc.STOPPED and rec[-1]["region"] == orc.REG_CT
        depth = rec[-1]["r"][2]
        assert R0 - 0.1 - 1e-4 <= depth <= R0 + 1e-4
        assert abs(depth - R0) < 0.01 * R0


@pytest.mark.parametrize("E", [70.0, 150.0])
@pytest.mark.parametrize("hz", [1.0, 2.0, 5.0])
def test_depth_dose_closed_form(E, hz):
    """IDD_k = ((R0-z_k)/alpha)^(1/p) - ((R0-z_{k+1})/alpha)^(1/p), independent of the voxel size."""
    R0 = ALPHA * E ** P
    nz = int(R0 / hz) + 3
    w = pencil_water(E, nz, hz)
    pb = oracle_problem(w, orc.default_params(flags=0), f32_params=False)
    e, tal = orc.dose_edep(pb, 1, 3)
    idd = grid(w, e).sum(axis=(1, 2))
    z = np.arange(nz + 1) * hz
    res = np.clip(R0 - z, 0, None)
    Ez = (res / ALPHA) ** (1 / P)
    expect = Ez[:-1] - Ez[1:]
    assert np.allclose(idd, expect, rtol=0, atol=1e-9 * E)
    assert abs(idd.sum() - E) < 1e-9 * E


# ------------------------------------------------------------------------------------------ P3

def highland_theta0(t, pv):
    return 13.6 / pv * math.sqrt(t) * (1 + 0.038 * math.log(t))


@pytest.mark.parametrize("n_steps", [1, 20])
def test_highland_thin_slab(n_steps):
    """2 mm of water at 100 MeV: projected exit-angle RMS = Highland, whatever the number of steps."""
    (E, mrad), = golden("highland_mrad")
    pv0 = (E * E + 2 * E * MP) / (E + MP)
    assert abs(pv0 - 190.37) < 0.01
    assert abs(highland_theta0(2.0 / 360.8, pv0) * 1e3 - mrad) < 2e-3
    N = 60000
    hz = 2.0 / n_steps
    w = pencil_water(E, n_steps, hz)
    pb = oracle_problem(w, orc.default_params(flags=flags(mcs=True)), f32_params=False)
    recs = orc.trace(pb, np.arange(N), N, 11, max_steps=64)
    ang = []
    for r in recs:
        last = r[-1]
        assert last["cause"] == orc.ESCAPED and last["region"] == orc.REG_CT
        assert len(r) == n_steps + 1        # entry drift + n_steps material steps
        ang.append((math.atan2(last["u"][0], last["u"][2]), math.atan2(last["u"][1], last["u"][2])))
    ang = np.array(ang)
    rms = math.sqrt(0.5 * (ang[:, 0].var() + ang[:, 1].var())) * 1e3
    assert abs(ang.mean()) < 5 * mrad * 1e-3 / math.sqrt(N)
    assert abs(rms - mrad) < 0.01 * mrad + 0.03          # golden value at entrance pv: +0.7% from the energy lost in the slab
    Emid = 0.5 * (E + ((ALPHA * E ** P - 2.0) / ALPHA) ** (1 / P))
    pvm = (Emid * Emid + 2 * Emid * MP) / (Emid + MP)
    if n_steps == 1:
        assert abs(rms - highland_theta0(2.0 / 360.8, pvm) * 1e3) < 0.006 * mrad
    # x and y projections uncorrelated and equal in variance (azimuth uniform)
    assert abs(np.corrcoef(ang[:, 0], ang[:, 1])[0, 1]) < 0.02
    assert abs(ang[:, 0].std() / ang[:, 1].std() - 1) < 0.02


def fermi_eyges_sigma(E0, dz=0.01):
    """Independent numerical Fermi-Eyges of the telescoped Highland form with start-of-step pv
    (the recipe SURVEY.md 8(c)-P3 states): sigma_x at the end of range."""
    R0 = ALPHA * E0 ** P
    n = int((R0 - 0.1) / dz)
    z = np.arange(n) * dz
    E = ((R0 - z) / ALPHA) ** (1 / P)
    pv = (E * E + 2 * E * MP) / (E + MP)
    t = (z + dz) / 360.8
    t0 = z / 360.8
    A = lambda x: np.where(x > 0, x * (1 + 0.038 * np.log(np.maximum(x, 1e-300))) ** 2, 0.0)
    T = (13.6 / pv) ** 2 * (A(t) - A(t0))       # angle variance gained in [z, z+dz]
    zend = n * dz
    return math.sqrt(np.sum(T * (zend - (z + 0.5 * dz)) ** 2))


@pytest.mark.parametrize("E,sig", golden("fe_sigma_mm"))
def test_lateral_sigma_at_end_of_range(E, sig):
    fe = fermi_eyges_sigma(E)
    assert abs(fe - sig) < 0.01 * sig                     # the golden number is reproducible from its recipe
    R0 = ALPHA * E ** P
    assert 0.018 * R0 < sig < 0.026 * R0                  # textbook ~2.2% of range
    N = 4000 if E < 200 else 1500
    hz = 2.0
    w = pencil_water(E, int(R0 / hz) + 3, hz)
    pb = oracle_problem(w, orc.default_params(flags=flags(mcs=True)), f32_params=False)
    recs = orc.trace(pb, np.arange(N), N, 5, max_steps=512)
    xy = np.array([(r[-1]["r"][0], r[-1]["r"][1]) for r in recs])
    assert all(r[-1]["cause"] == orc.STOPPED for r in recs)
    s = math.sqrt(0.5 * (xy[:, 0].var() + xy[:, 1].var()))
    assert abs(s - sig) < 0.05 * sig + 3 * sig / math.sqrt(2 * N)
    assert abs(xy.mean()) < 5 * sig / math.sqrt(N)


def test_scatter_rotation_invariants():
    """Each step turns the direction by exactly theta = theta0 sqrt(-2 ln u0) (dot product), keeps it unit,
    and moves along the OLD direction."""
    E = 100.0
    w = pencil_water(E, 30, 2.0)
    pb = oracle_problem(w, orc.default_params(flags=flags(mcs=True)), f32_params=False)
    seed = 21
    recs = orc.trace(pb, np.arange(50), 50, seed, max_steps=256)
    checked = 0
    for r in recs:
        hid = int(r[0]["hid"])
        t_rad = 0.0
        for k in range(1, len(r)):
            a, b = r[k - 1], r[k]
            if b["cause"] != orc.CONT:
                break
            assert abs(np.linalg.norm(b["u"]) - 1) < 1e-14
            s = b["s"]
            # moved along the old direction (faces snap one coordinate, so compare the free ones loosely)
            assert np.allclose(b["r"], a["r"] + s * a["u"], atol=1e-9)
            x = orc.philox4x32_10([hid & 0xFFFFFFFF, hid >> 32, int(b["step"]), 0], [seed, 0])
            u0 = orc.u01(x[0])
            Em = 0.5 * (b["E_before"] + b["E_after"])
            pv = (Em * Em + 2 * Em * MP) / (Em + MP)
            A = lambda t: t * (1 + 0.038 * math.log(t)) ** 2 if t > 0 else 0.0
            tp = t_rad + s / 360.8
            theta = 13.6 / pv * math.sqrt(A(tp) - A(t_rad)) * math.sqrt(-2 * math.log(u0))
            t_rad = tp
            cosang = float(np.dot(a["u"], b["u"]))
            assert abs(cosang - math.cos(theta)) < 1e-12
            checked += 1
    assert checked > 1000


# ------------------------------------------------------------------------------------------ P4

def test_range_straggling_bohr():
    (E, bohr), = golden("straggle_mm")
    (_, bortfeld), = golden("bortfeld_mm")
    R0 = ALPHA * E ** P
    assert abs(0.012 * (R0 / 10) ** 0.935 * 10 - bortfeld) < 0.01
    assert abs(bohr - bortfeld) < 0.1 * bortfeld
    # independent Bohr integral: sigma_R^2 = int sigma_E^2'(E) / S(E)^2 dz
    z = np.arange(0, R0 - 0.1, 0.01)
    Ez = ((R0 - z) / ALPHA) ** (1 / P)
    g = 1 + Ez / MP
    b2 = 1 - 1 / g ** 2
    dvar = 0.015692 * 0.5551 * g ** 2 * (1 - b2 / 2)        # MeV^2 per mm
    S = Ez ** (1 - P) / (ALPHA * P)
    integral = math.sqrt(np.sum(dvar / S ** 2) * 0.01)
    assert abs(integral - bohr) < 0.02 * bohr
    N = 6000
    w = pencil_water(E, int(R0) + 8, 1.0)
    pb = oracle_problem(w, orc.default_params(flags=flags(straggle=True)), f32_params=False)
    recs = orc.trace(pb, np.arange(N), N, 9, max_steps=512)
    depth = np.array([r[-1]["r"][2] for r in recs])
    assert all(r[-1]["cause"] == orc.STOPPED for r in recs)
    assert abs(depth.std() - bohr) < 0.05 * bohr + 3 * bohr / math.sqrt(2 * N)
    assert abs(depth.std() - bortfeld) < 0.1 * bortfeld
    assert abs(depth.mean() - R0) < 0.01 * R0


def test_sigma_E_check_value():
    """C4-4 check value: one 1 mm water step at 100 MeV straggles by sigma_E = 0.0984 MeV."""
    (E, sE), = golden("sigma_E_MeV")
    N = 40000
    w = pencil_water(E, 1, 1.0)
    pb = oracle_problem(w, orc.default_params(flags=flags(straggle=True)), f32_params=False)
    recs = orc.trace(pb, np.arange(N), N, 17, max_steps=8)
    Ea = np.array([r[1]["E_after"] for r in recs])
    Ebar = ((ALPHA * E ** P - 1.0) / ALPHA) ** (1 / P)
    assert abs(Ea.std() - sE) < 0.01 * sE + 3 * sE / math.sqrt(2 * N)
    assert abs(Ea.mean() - Ebar) < 4 * sE / math.sqrt(N)


# ------------------------------------------------------------------------------------------ P5

@pytest.mark.parametrize("E,surv", golden("survival"))
def test_nuclear_survival(E, surv):
    R0 = ALPHA * E ** P
    assert abs(1 / (1 + 0.0012 * R0) - surv) < 1e-4
    N = 20000
    hz = 2.0
    w = pencil_water(E, int(R0 / hz) + 3, hz)
    pb = oracle_problem(w, orc.default_params(flags=flags(nuclear=True)), f32_params=False)
    _, tal = orc.dose_edep(pb, N, 13)
    assert tal.n_nuclear + tal.n_stopped_ct == N
    got = tal.n_stopped_ct / N
    # the last R_cut of range is not traversed: survival to R_cut residual = (1+beta R_cut)/(1+beta R0)
    expect = (1 + 0.0012 * 0.1) / (1 + 0.0012 * R0)
    assert abs(got - expect) < 4 * math.sqrt(surv * (1 - surv) / N)
    assert abs(got - surv) < 4 * math.sqrt(surv * (1 - surv) / N) + 2e-4


def test_nuclear_depth_profile_linear_in_residual_range():
    E = 150.0
    R0 = ALPHA * E ** P
    N = 40000
    w = pencil_water(E, int(R0 / 2.0) + 3, 2.0)
    pb = oracle_problem(w, orc.default_params(flags=flags(nuclear=True)), f32_params=False)
    recs = orc.trace(pb, np.arange(N), N, 4, max_steps=512)
    zs = np.array([r[-1]["r"][2] for r in recs if r[-1]["cause"] == orc.NUCLEAR])
    # N(z)/N0 = (1 + beta (R0 - z)) / (1 + beta R0): fraction removed before depth z (to the voxel resolution)
    for zq in (40.0, 80.0, 120.0):
        frac = 1 - (1 + 0.0012 * (R0 - zq)) / (1 + 0.0012 * R0)
        got = np.mean(zs < zq - 1e-9) * len(zs) / N
        assert abs(got - frac) < 4 * math.sqrt(frac / N) + 0.0012 * 2.0


# ------------------------------------------------------------------------------------------ P6

@pytest.mark.parametrize("case", ["config1", "rs_ap", "hetero"])
def test_energy_bookkeeping(case):
    if case == "config1":
        w = wl.config1()
    elif case == "rs_ap":
        w = wl.small_water(n=(20, 20, 60), energy=150.0, sigma=4.0, with_aperture=True, rs_wet=45.0, n_spots=3)
    else:
        w = wl.small_water(n=(12, 12, 30), energy=90.0, sigma=5.0, with_aperture=True, n_spots=2)
        rng = np.random.default_rng(5)
        w["ct"]["hu"] = rng.integers(-1000, 1500, size=w["ct"]["hu"].shape).astype(np.int16)
    pb = oracle_problem(w)
    N = 3000
    e, tal = orc.dose_edep(pb, N, 2)
    t = tal.as_dict()
    total = t["dep_ct"] + t["dep_rs"] + t["dep_brass"] + t["escaped"] + t["removed"]
    assert abs(total - t["incident"]) <= 1e-6 * t["incident"]
    assert abs(total - t["incident"]) <= 1e-10 * t["incident"]
    assert t["n_stopped_ct"] + t["n_stopped_rs"] + t["n_stopped_brass"] + t["n_nuclear"] + t["n_escaped"] == N
    assert abs(e.sum() - t["dep_ct"]) <= 1e-10 * max(t["dep_ct"], 1.0)
    assert (e >= 0).all()


# ------------------------------------------------------------------------------------------ P7

def closed_block(E, sigma=3.0, all_flags=True):
    w = wl.small_water(n=(20, 20, 30), energy=E, sigma=sigma, with_aperture=True, opening_radius=3.0)
    w["beams"][0]["aperture"]["open"][:] = 0
    return w


@pytest.mark.parametrize("E", [71.3, 100.0, 150.0])
def test_closed_block_stops_everything_up_to_150MeV(E):
    """30 mm brass blocks protons up to about 155 MeV -> zero fluence behind a closed block."""
    w = closed_block(E)
    pb = oracle_problem(w)
    N = 2000
    e, tal = orc.dose_edep(pb, N, 8)
    assert tal.dep_ct == 0.0 and not e.any()
    assert tal.n_stopped_ct == 0
    assert tal.n_stopped_brass + tal.n_nuclear + tal.n_escaped == N
    assert tal.n_stopped_brass > 0.5 * N


def test_block_range_limit_is_155MeV():
    """Loss only: 155 MeV just stops in 30 mm brass, 156 MeV just gets out (RSP 5.523 from P:L81)."""
    for E, through in ((154.9, False), (155.2, True)):
        w = closed_block(E, sigma=0.0)
        pb = oracle_problem(w, orc.default_params(flags=0), f32_params=False)
        rec = orc.trace(pb, [0], 1, 1)[0]
        got_through = any(q["region"] == orc.REG_CT for q in rec)
        assert got_through == through


@pytest.mark.parametrize("E,Eexit", golden("brass_exit"))
def test_brass_exit_energy(E, Eexit):
    w = closed_block(E, sigma=0.0)
    pb = oracle_problem(w, orc.default_params(flags=0), f32_params=False)
    rec = orc.trace(pb, [0], 1, 1)[0]
    brass = rec[rec["region"] == orc.REG_AP_BRASS]
    assert len(brass) >= 30                                # s_ap = 1 mm steps (+ f_R refinement near end of range)
    assert len(brass) == 30 or E < 200
    assert abs(brass["s"].sum() - 30.0) < 1e-12
    assert abs(brass[-1]["E_after"] - Eexit) < 0.01
    if E == 161.5:
        assert abs(ALPHA * brass[-1]["E_after"] ** P - 12.50) < 0.01     # residual range


# ------------------------------------------------------------------------------------------ P8

def test_config1_open_fraction():
    """MCS off: a history passes iff it is sampled inside the 10 mm disc; fraction 1 - exp(-r^2/2 sigma^2)."""
    w = wl.config1()
    pb = oracle_problem(w, orc.default_params(flags=0))
    N = 20000
    _, tal = orc.dose_edep(pb, N, 1)
    p = 1 - math.exp(-10.0 ** 2 / (2 * 4.0 ** 2))
    assert abs(p - 0.95606) < 1e-5
    passed = tal.n_stopped_ct
    assert tal.n_stopped_brass == N - passed
    assert abs(passed - N * p) < 3 * math.sqrt(N * p * (1 - p)) + 0.002 * N   # + pixelation of the disc edge


def test_source_gaussian_moments():
    w = wl.small_water(n=(40, 40, 4), h=(2.0, 2.0, 2.0), energy=100.0, sigma=4.0)
    w["beams"][0]["spots"][0, 0:2] = (3.0, -2.0)
    pb = oracle_problem(w, orc.default_params(flags=0))
    N = 20000
    recs = orc.trace(pb, np.arange(N), N, 6, max_steps=16)
    xy = np.array([r[0]["r"][:2] for r in recs])
    assert abs(xy[:, 0].mean() - 3.0) < 4 * 4.0 / math.sqrt(N)
    assert abs(xy[:, 1].mean() + 2.0) < 4 * 4.0 / math.sqrt(N)
    assert abs(xy[:, 0].std() - 4.0) < 4 * 4.0 / math.sqrt(2 * N)
    assert abs(xy[:, 1].std() - 4.0) < 4 * 4.0 / math.sqrt(2 * N)
    assert abs(np.corrcoef(xy.T)[0, 1]) < 0.03


# ------------------------------------------------------------------------------------------ P9

@pytest.mark.parametrize("E,Eexit", golden("rs_exit"))
def test_range_shifter_exit_energy(E, Eexit):
    w = wl.small_water(n=(5, 5, 10), h=(100.0, 100.0, 50.0), energy=E, sigma=0.0, rs_wet=45.0)
    pb = oracle_problem(w, orc.default_params(flags=0), f32_params=False)
    rec = orc.trace(pb, [0], 1, 1)[0]
    rs = rec[rec["region"] == orc.REG_RS]
    assert len(rs) == 45 and abs(rs["s"].sum() - 45.0) < 1e-12
    assert abs(rs[-1]["E_after"] - Eexit) < 1e-3


def test_range_shifter_absorbs_below_74MeV():
    for E, through in ((74.0, False), (74.5, True)):
        w = wl.small_water(n=(5, 5, 10), h=(100.0, 100.0, 50.0), energy=E, sigma=0.0, rs_wet=45.0)
        pb = oracle_problem(w, orc.default_params(flags=0), f32_params=False)
        rec = orc.trace(pb, [0], 1, 1)[0]
        if through:
            assert any(q["region"] == orc.REG_CT for q in rec)
        else:
            assert rec[-1]["cause"] == orc.STOPPED and rec[-1]["region"] == orc.REG_RS
