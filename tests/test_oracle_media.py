"""Pins of the parts of the oracle that only matter outside homogeneous water on axis (VERDICT
round 1, "what's weak" 1): the brass constants, media with rho != RSP != scattering power, the range
scenario touching RSP only (R12), the locally absorbed fraction of a nuclear event, the orientation
of the opening bitmap, state carried from one medium into the next (t_rad, tau, the step counter that keys the Philox
stream), and the face crossing of a history that scatters back on the face (C4-8/9, R8).

Expectations are closed forms evaluated here (Highland, Bohr, exponential attenuation, Gaussian mass over a rectangle),
golden values from tests/golden/physics_pins.txt with their derivation, and hand-traced discrete outcomes on a 4^3 grid
with injected uniforms.  Nothing compares the oracle with itself or with the CUDA path.
"""
import math

import numpy as np
import pytest

from oracle import vpmc_oracle as orc
from paper_2307_01416_b200 import workloads as wl
from tests.helpers import oracle_problem, read_golden

ALPHA, P = 0.022, 1.77
MP = 938.272
X0_W, X0_BRASS = 360.8, 14.94
BETA = 0.0012


def golden(kind):
    return [(float(r[1]), float(r[2])) for r in read_golden("physics_pins.txt") if r[0] == kind]


def flags(**on):
    f = 0
    if on.get("mcs"): f |= orc.FLAG_MCS
    if on.get("straggle"): f |= orc.FLAG_STRAGGLE
    if on.get("nuclear"): f |= orc.FLAG_NUCLEAR
    return f


def pv_of(E):
    return (E * E + 2 * E * MP) / (E + MP)


def highland_A(t):
    return t * (1 + 0.038 * math.log(t)) ** 2 if t > 0 else 0.0


def energy_after(E, wet):
    return ((ALPHA * E ** P - wet) / ALPHA) ** (1 / P)


# ------------------------------------------------------------------------------------------ brass (C0, C4-4, C4-7)

def brass_slab(E, thickness):
    """A closed brass block of the given thickness in front of a wide water box: every history crosses the brass."""
    w = wl.small_water(n=(5, 5, 4), h=(400.0, 400.0, 5.0), energy=E, sigma=0.0, with_aperture=True)
    w["beams"][0]["aperture"]["open"][:] = 0
    w["beams"][0]["aperture"]["T"] = np.float32(thickness)
    return w


@pytest.mark.parametrize("n_steps", [1, 2, 20])
def test_highland_thin_slab_of_brass(n_steps):
    """2 mm of brass (X0 = 14.94 mm) at 200 MeV: exit projected-angle RMS = Highland with t = 2 / 14.94, whatever the
    number of steps.  With water's radiation length the angle would be 5.5 times smaller."""
    (E, mrad), = golden("highland_brass_mrad")
    t = 2.0 / X0_BRASS
    assert abs(13.6 / pv_of(E) * math.sqrt(t) * (1 + 0.038 * math.log(t)) * 1e3 - mrad) < 2e-3
    N = 40000
    pb = oracle_problem(brass_slab(E, 2.0), orc.default_params(flags=flags(mcs=True), s_ap=2.0 / n_steps), f32_params=False)
    recs = orc.trace(pb, np.arange(N), N, 23, max_steps=64)
    ang = []
    for r in recs:
        b = r[r["region"] == orc.REG_AP_BRASS]
        # a scattered history needs a last short step to reach the exit plane (depth gained per step = s u_w < s)
        assert len(b) in (n_steps, n_steps + 1) and 0.0 <= b["s"].sum() - 2.0 < 1e-2
        u = b[-1]["u"]
        ang.append((math.atan2(u[0], u[2]), math.atan2(u[1], u[2])))
    ang = np.array(ang)
    rms = math.sqrt(0.5 * (ang[:, 0].var() + ang[:, 1].var())) * 1e3
    Emid = 0.5 * (E + energy_after(E, 2.0 * 5.523))           # pv at the mean energy of the slab (single step: exact)
    expect = 13.6 / pv_of(Emid) * math.sqrt(highland_A(t)) * 1e3
    assert abs(expect - mrad) < 0.02 * mrad
    assert abs(rms - expect) < 0.006 * expect + 3 * expect / math.sqrt(2 * N)
    assert abs(ang.mean()) < 5 * mrad * 1e-3 / math.sqrt(N)


def test_sigma_E_of_one_brass_step():
    """C4-4 in brass: one 1 mm step at 200 MeV straggles by sqrt(k_bohr * 0.457 * 8.5 * gamma^2 (1 - beta^2 / 2))."""
    (E, sE), = golden("sigma_E_brass_MeV")
    g = 1 + E / MP
    assert abs(math.sqrt(0.015692 * 0.457 * 8.5 * g * g * (1 - 0.5 * (1 - 1 / g ** 2))) - sE) < 1e-4
    N = 40000
    pb = oracle_problem(brass_slab(E, 1.0), orc.default_params(flags=flags(straggle=True)), f32_params=False)
    recs = orc.trace(pb, np.arange(N), N, 29, max_steps=16)
    Ea = []
    for r in recs:
        b = r[r["region"] == orc.REG_AP_BRASS]
        assert len(b) == 1
        Ea.append(b[0]["E_after"])
    Ea = np.array(Ea)
    Ebar = energy_after(E, 5.523)
    assert abs(Ea.std() - sE) < 0.01 * sE + 3 * sE / math.sqrt(2 * N)
    assert abs(Ea.mean() - Ebar) < 4 * sE / math.sqrt(N)


def test_nuclear_loss_in_brass_scales_with_its_density():
    """C4-6 in brass: tau grows by beta / (1 + beta R) * rho_rel * s with rho_rel = 8.5 and s the GEOMETRIC step."""
    E, T = 200.0, 10.0
    N = 40000
    pb = oracle_problem(brass_slab(E, T), orc.default_params(flags=flags(nuclear=True)), f32_params=False)
    recs = orc.trace(pb, np.arange(N), N, 31, max_steps=64)
    n_nuc = sum(1 for r in recs if r[-1]["cause"] == orc.NUCLEAR and r[-1]["region"] == orc.REG_AP_BRASS)
    # closed form: R(z) = R0 - 5.523 z  ->  tau = (8.5 / 5.523) ln((1 + beta R0) / (1 + beta (R0 - 5.523 T)))
    R0 = ALPHA * E ** P
    tau = 8.5 / 5.523 * math.log((1 + BETA * R0) / (1 + BETA * (R0 - 5.523 * T)))
    p = 1 - math.exp(-tau)
    assert 0.05 < p < 0.12
    assert abs(n_nuc / N - p) < 4 * math.sqrt(p * (1 - p) / N) + 0.004 * p      # + start-of-step rule over 10 steps


# ------------------------------------------------------------------------------------------ rho != RSP != xsp (C5, R12)

MEDIUM = {"hu": np.array([0.0, 1000.0]), "rsp": np.array([1.0, 1.6]), "rho": np.array([1.0, 3.0]),
          "xsp": np.array([1.0, 0.4])}            # HU 500 -> RSP 1.3, rho 2.0, scattering power 0.7


def medium_column(E, nz, hz):
    w = wl.small_water(n=(5, 5, nz), h=(400.0, 400.0, hz), energy=E, sigma=0.0)
    w["ct"]["hu"][:] = 500
    w["calib"] = dict(MEDIUM)
    return w


def test_medium_calibration_nodes():
    assert orc.calib_eval(MEDIUM, 500.0) == (1.3, 2.0, 0.7)


def test_nuclear_survival_follows_density_not_rsp():
    """Survival to the end of range in a medium with rho_rel = 2, RSP = 1.3:
    ((1 + beta R_cut) / (1 + beta R0))^(rho_rel / RSP); without the density factor the exponent would be 1 / RSP."""
    E = 150.0
    R0 = ALPHA * E ** P
    N = 20000
    pb = oracle_problem(medium_column(E, int(R0 / 1.3 / 2.0) + 3, 2.0), orc.default_params(flags=flags(nuclear=True)), f32_params=False)
    _, tal = orc.dose_edep(pb, N, 37)
    assert tal.n_nuclear + tal.n_stopped_ct == N
    expect = ((1 + BETA * 0.1) / (1 + BETA * R0)) ** (2.0 / 1.3)
    assert abs(expect - 0.7677) < 1e-4
    assert abs(tal.n_stopped_ct / N - expect) < 4 * math.sqrt(expect * (1 - expect) / N) + 1e-3


@pytest.mark.parametrize("rsp_scale", [1.0, 1.5])
def test_one_step_nuclear_probability_ignores_the_range_scenario(rsp_scale):
    """One 2 mm voxel layer: P(nuclear) = 1 - exp(-beta / (1 + beta R0) * rho_rel * s), whatever rsp_scale (the
    range scenario scales the RSP; density stays nominal, R12)."""
    E = 100.0
    N = 200000
    pb = oracle_problem(medium_column(E, 1, 2.0), orc.default_params(flags=flags(nuclear=True)), f32_params=False)
    _, tal = orc.dose_edep(pb, N, 41, orc.scenario(rsp_scale=rsp_scale))
    p = 1 - math.exp(-BETA / (1 + BETA * ALPHA * E ** P) * 2.0 * 2.0)
    assert tal.n_nuclear + tal.n_escaped == N
    assert abs(tal.n_nuclear - N * p) < 4 * math.sqrt(N * p)


@pytest.mark.parametrize("rsp_scale", [1.0, 1.5])
def test_scattering_follows_the_scattering_power(rsp_scale):
    """2 mm of the medium at 100 MeV: theta0 = Highland with t = 2 * xsp / X0_w (xsp = 0.7), not RSP (1.3) nor rho (2);
    the range scenario leaves it unchanged up to the mid-step energy."""
    E = 100.0
    N = 40000
    pb = oracle_problem(medium_column(E, 1, 2.0), orc.default_params(flags=flags(mcs=True)), f32_params=False)
    recs = orc.trace(pb, np.arange(N), N, 43, orc.scenario(rsp_scale=rsp_scale), max_steps=8)
    ang = np.array([(math.atan2(r[-1]["u"][0], r[-1]["u"][2]), math.atan2(r[-1]["u"][1], r[-1]["u"][2])) for r in recs])
    assert all(len(r) == 2 for r in recs)
    rms = math.sqrt(0.5 * (ang[:, 0].var() + ang[:, 1].var()))
    Emid = 0.5 * (E + energy_after(E, 2.0 * 1.3 * rsp_scale))
    expect = 13.6 / pv_of(Emid) * math.sqrt(highland_A(2.0 * 0.7 / X0_W))
    assert abs(rms - expect) < 0.004 * expect + 3 * expect / math.sqrt(2 * N)
    wrong = 13.6 / pv_of(Emid) * math.sqrt(highland_A(2.0 * 1.3 / X0_W))
    assert abs(rms - wrong) > 0.2 * expect


def test_straggling_follows_density():
    """C4-4 in a CT voxel: za rho = za_w * rho_rel, so one 1 mm step of the medium (rho_rel = 2) at 100 MeV straggles by
    sqrt(2) times the water check value 0.0984 MeV (golden `sigma_E_MeV`), not by sqrt(RSP)."""
    (E, sE_w), = [(float(r[1]), float(r[2])) for r in read_golden("physics_pins.txt") if r[0] == "sigma_E_MeV"]
    sE = sE_w * math.sqrt(2.0)
    N = 40000
    pb = oracle_problem(medium_column(E, 1, 1.0), orc.default_params(flags=flags(straggle=True)), f32_params=False)
    recs = orc.trace(pb, np.arange(N), N, 45, max_steps=8)
    Ea = np.array([r[1]["E_after"] for r in recs])
    assert abs(Ea.std() - sE) < 0.01 * sE + 3 * sE / math.sqrt(2 * N)
    assert abs(Ea.mean() - energy_after(E, 1.3)) < 4 * sE / math.sqrt(N)


def test_energy_loss_follows_rsp_times_scale():
    """Loss only: exit energy of 10 mm of the medium = E(R0 - 10 * 1.3 * scale)."""
    for scale in (1.0, 0.965, 1.035):
        pb = oracle_problem(medium_column(120.0, 5, 2.0), orc.default_params(flags=0), f32_params=False)
        rec = orc.trace(pb, [0], 1, 1, orc.scenario(rsp_scale=scale))[0]
        assert rec[-1]["cause"] == orc.ESCAPED
        assert abs(rec[-1]["E_after"] - energy_after(120.0, 10.0 * 1.3 * scale)) < 1e-9


# ------------------------------------------------------------------------------------------ gamma_loc (C0, C4-6)

def test_locally_absorbed_fraction_of_a_nuclear_event():
    """C4-6: a nuclear event deposits gamma_loc = 0.6 of the remaining energy locally and removes 0.4 of it."""
    E, N, seed = 150.0, 4000, 47
    R0 = ALPHA * E ** P
    w = wl.small_water(n=(5, 5, int(R0 / 2.0) + 3), h=(400.0, 400.0, 2.0), energy=E, sigma=0.0)
    pb = oracle_problem(w, orc.default_params(flags=flags(nuclear=True)), f32_params=False)
    _, tal = orc.dose_edep(pb, N, seed)
    recs = orc.trace(pb, np.arange(N), N, seed, max_steps=256)
    E_at_event = sum(float(r[-1]["E_after"]) for r in recs if r[-1]["cause"] == orc.NUCLEAR)
    lost_along = sum(float((r["E_before"] - r["E_after"])[r["region"] == orc.REG_CT].sum()) for r in recs)
    assert tal.n_nuclear > 400
    assert abs(tal.removed - 0.4 * E_at_event) < 1e-9 * E_at_event
    assert abs(tal.dep_ct - (lost_along + 0.6 * E_at_event)) < 1e-9 * tal.incident


# ------------------------------------------------------------------------------------------ opening bitmap orientation (C4)

def slot_problem(transposed):
    """A 2 x 6 mm slot off centre in a NON-square bitmap (96 x 128 pixels of 0.1 mm), spot at (3, 0), sigma 3 mm."""
    w = wl.small_water(n=(40, 40, 10), h=(2.0, 2.0, 2.0), energy=100.0, sigma=3.0, with_aperture=True)
    nx, ny = (128, 96) if transposed else (96, 128)
    u0, v0 = -0.05 * nx, -0.05 * ny
    xc = u0 + (np.arange(nx) + 0.5) * 0.1
    yc = v0 + (np.arange(ny) + 0.5) * 0.1
    X, Y = np.meshgrid(xc, yc, indexing="xy")             # [iy, ix]
    if transposed:
        op = (X > -4) & (X < 2) & (Y > 2) & (Y < 4)
    else:
        op = (X > 2) & (X < 4) & (Y > -4) & (Y < 2)
    ap = w["beams"][0]["aperture"]
    ap["open"] = op.astype(np.uint8)
    ap["u0"], ap["v0"] = np.float32(u0), np.float32(v0)
    w["beams"][0]["spots"][0, 0:2] = (3.0, 0.0)
    return w


@pytest.mark.parametrize("transposed", [False, True])
def test_asymmetric_slot_opening(transposed):
    """MCS off: a history passes iff it is sampled inside the slot: N * Gaussian mass over the rectangle; the mass of the
    transposed slot is three times smaller, so a swapped (ix, iy) lookup fails both cases."""
    Phi = lambda x: 0.5 * (1 + math.erf(x / math.sqrt(2)))
    if transposed:
        p = (Phi((2 - 3) / 3) - Phi((-4 - 3) / 3)) * (Phi(4 / 3) - Phi(2 / 3))
        assert abs(p - 0.05800) < 1e-5
    else:
        p = (Phi((4 - 3) / 3) - Phi((2 - 3) / 3)) * (Phi(2 / 3) - Phi(-4 / 3))
        assert abs(p - 0.17137) < 1e-5
    N = 20000
    pb = oracle_problem(slot_problem(transposed), orc.default_params(flags=0))
    _, tal = orc.dose_edep(pb, N, 53)
    passed = N - tal.n_stopped_brass
    assert passed == tal.n_escaped + tal.n_stopped_ct
    assert abs(passed - N * p) < 4 * math.sqrt(N * p * (1 - p))


# ------------------------------------------------------------------------------------------ state carried across media (C4 last paragraph, C1)

def rs_then_water(E, flags_, hz=2.0, nz=100):
    w = wl.small_water(n=(5, 5, nz), h=(400.0, 400.0, hz), energy=E, sigma=0.0, rs_wet=45.0)
    return oracle_problem(w, orc.default_params(flags=flags_), f32_params=False)


def test_t_rad_is_carried_from_the_range_shifter_into_the_ct():
    """First 2 mm CT step behind a 45 mm WET range shifter: theta0^2 = (Es/pv)^2 [A(t + dt) - A(t)], t = 45 / 360.8;
    a fresh t_rad = 0 would give A(dt): 1.195 times smaller in theta0 (golden `carried_ratio`)."""
    (E, ratio), = golden("carried_ratio")
    t0, dt = 45.0 / X0_W, 2.0 / X0_W
    assert abs(math.sqrt((highland_A(t0 + dt) - highland_A(t0)) / highland_A(dt)) - ratio) < 1e-4
    N = 30000
    pb = rs_then_water(E, flags(mcs=True))
    recs = orc.trace(pb, np.arange(N), N, 59, max_steps=256)
    th2 = []
    for r in recs:
        k = int(np.argmax(r["region"] == orc.REG_CT))
        # the scattered path through the slab is a little longer than its thickness
        assert r[k - 1]["region"] == orc.REG_VAC and 0.0 <= r[k - 1]["t_rad"] - t0 < 1e-2 * t0
        c = float(np.dot(r[k - 1]["u"], r[k]["u"]))
        th2.append(2.0 * (1.0 - c))                        # theta^2 for small theta
        assert abs(r[k]["t_rad"] - (r[k - 1]["t_rad"] + r[k]["s"] / X0_W)) < 1e-12
    E1 = energy_after(E, 45.0)
    Emid = 0.5 * (E1 + energy_after(E1, 2.0))
    theta0 = 13.6 / pv_of(Emid) * math.sqrt(highland_A(t0 + dt) - highland_A(t0))
    got = math.sqrt(0.5 * np.mean(th2))                    # E[theta^2] = 2 theta0^2
    assert abs(got - theta0) < 0.005 * theta0 + 3 * theta0 / math.sqrt(2 * N)


def test_tau_is_carried_from_the_range_shifter_into_the_ct():
    """Nuclear only, 150 MeV through the 45 mm WET range shifter and then water to the end of range: the optical depth
    keeps accumulating against the SAME threshold, so P(event in the CT | survived the slab) = 1 - exp(-tau_ct); a tau
    reset at the CT entry would give 1 - exp(-(tau_ct - tau_rs))."""
    E, N = 150.0, 30000
    R0 = ALPHA * E ** P
    pb = rs_then_water(E, flags(nuclear=True))
    recs = orc.trace(pb, np.arange(N), N, 61, max_steps=256)
    n_rs = sum(1 for r in recs if r[-1]["cause"] == orc.NUCLEAR and r[-1]["region"] == orc.REG_RS)
    n_ct = sum(1 for r in recs if r[-1]["cause"] == orc.NUCLEAR and r[-1]["region"] == orc.REG_CT)
    n_stop = sum(1 for r in recs if r[-1]["cause"] == orc.STOPPED)
    assert n_rs + n_ct + n_stop == N
    p_rs = 1 - (1 + BETA * (R0 - 45.0)) / (1 + BETA * R0)
    p_ct = 1 - (1 + BETA * 0.1) / (1 + BETA * (R0 - 45.0))
    assert abs(n_rs / N - p_rs) < 4 * math.sqrt(p_rs / N) + 2e-4
    assert abs(n_ct / (N - n_rs) - p_ct) < 4 * math.sqrt(p_ct / N) + 5e-4
    tau_rs = math.log((1 + BETA * R0) / (1 + BETA * (R0 - 45.0)))
    wrong = 1 - math.exp(-(-math.log(1 - p_ct) - tau_rs))
    assert abs(n_ct / (N - n_rs) - wrong) > 0.03


def test_step_counter_counts_vacuum_drifts_and_keys_the_stream():
    """C3: a vacuum drift uses no random numbers but increments the step counter; C1: the block of step k is
    Philox(hid, k, purpose 0).  On axis, loss + straggling: drift 0, 45 range-shifter steps 1..45, drift 46, 30 opening
    steps 47..76, CT-entry drift 77, first CT step 78, whose straggling must come from block 78."""
    w = wl.small_water(n=(5, 5, 60), h=(400.0, 400.0, 2.0), energy=150.0, sigma=0.0, with_aperture=True, rs_wet=45.0,
                       opening_radius=3.0)
    pb = oracle_problem(w, orc.default_params(flags=flags(straggle=True)), f32_params=False)
    seed = 67
    for hid, r in zip((0, 5), orc.trace(pb, [0, 5], 10, seed, max_steps=256)):
        assert list(r["step"]) == list(range(len(r)))
        reg = list(r["region"][:79])
        assert reg == [orc.REG_VAC] + [orc.REG_RS] * 45 + [orc.REG_VAC] + [orc.REG_AP_OPEN] * 30 + [orc.REG_VAC] + [orc.REG_CT]
        q = r[78]
        x = orc.philox4x32_10([hid, 0, 78, 0], [seed, 0])
        z0 = math.sqrt(-2 * math.log(orc.u01(x[2]))) * math.cos(2 * math.pi * orc.u01(x[3]))
        Ebar = energy_after(q["E_before"], q["s"])
        g = 1 + 0.5 * (q["E_before"] + Ebar) / MP
        sE = math.sqrt(0.015692 * 0.5551 * q["s"] * g * g * (1 - 0.5 * (1 - 1 / g ** 2)))
        assert abs((q["E_after"] - Ebar) + sE * z0) < 1e-9
        y = orc.philox4x32_10([hid, 0, 77, 0], [seed, 0])          # the neighbouring block does not reproduce it
        z1 = math.sqrt(-2 * math.log(orc.u01(y[2]))) * math.cos(2 * math.pi * orc.u01(y[3]))
        assert abs((q["E_after"] - Ebar) + sE * z1) > 1e-6


# ------------------------------------------------------------------------------------------ C4-8/9: scattering back on a face (R8)

def rot_small(axis, eps):
    c, s = math.cos(eps), math.sin(eps)
    if axis == 0:         # beam direction (sin eps, 0, cos eps) in the CT frame
        return np.array([[c, 0, s], [0, 1, 0], [-s, 0, c]])
    return np.array([[1, 0, 0], [0, c, s], [0, -s, c]])       # (0, sin eps, cos eps)


@pytest.mark.parametrize("axis", [0, 1])
@pytest.mark.parametrize("sgn", [+1, -1])
def test_hand_traced_scatter_back_on_a_face(axis, sgn):
    """4^3 grid of 1 x 1 x 10 mm voxels, MCS only, injected uniforms.  The history enters the z = 0 face 1 um short of
    the lateral face at coordinate 0, travelling towards it at 2 mrad, and reaches it after 0.5 mm.  The injected block
    of that step (u0 = 2^-24: theta = 5.8 theta0 = 11.5 mrad; u1 = 0.5: azimuth pi, back towards the axis) reverses the
    sign of that direction cosine ON the step that ends on the face.  C4-8 moves along the OLD direction and C4-9
    advances the index of the face that was reached: the history is now in the neighbour voxel, on its near face,
    heading back; the next step has zero length and re-crosses; the third runs to the z face inside the first voxel.
    (Deciding the crossing from the direction AFTER the rotation would instead put it one voxel the other way, on the
    far face.)"""
    eps, delta = 2e-3 * sgn, 1e-3
    origin = [-2.0, -2.0, 0.0]
    ct = {"n": (4, 4, 4), "h": (1.0, 1.0, 10.0), "origin": tuple(origin), "hu": np.zeros((4, 4, 4), dtype=np.int16)}
    xs = [0.3, 0.3]                                      # the other lateral coordinate sits mid-voxel (index 2)
    xs[axis] = -sgn * delta * math.cos(eps)               # entry at lateral coordinate -sgn * delta (iso on the z = 0 face)
    beam = {"iso": np.zeros(3), "rot": rot_small(axis, eps), "spots": np.array([[xs[0], xs[1], 100.0, 1.0, 0.0]]),
            "rs_wet": 0.0, "rs_face": 190.0, "aperture": None}
    pb = orc.Problem(ct=ct, calib=wl.calibration(), beams=[beam], params=orc.default_params(flags=flags(mcs=True)))
    tiny = 2.0 ** -24
    inject = [[0.5, 0.25, 0.5, 0.5], [tiny, 0.5 + tiny, 0.5, 0.5], [0.5, 0.25, 0.5, 0.5], [0.5, 0.25, 0.5, 0.5]]
    with orc.injected_uniforms(inject):
        r = orc.trace(pb, [0], 1, 1, max_steps=64)[0]
    first = 1 if sgn > 0 else 2                           # voxel index on `axis` at entry: [-1, 0) or [0, 1)
    nb = first + sgn
    other = 1 - axis
    assert r[0]["region"] == orc.REG_VAC and r[1]["region"] == orc.REG_CT
    assert abs(r[0]["r"][axis] + sgn * delta) < 1e-12 and r[0]["r"][2] == 0.0
    # step 1: reaches the face after ~0.5 mm, direction cosine changes sign
    assert r[1]["ivox"][axis] == first and r[1]["ivox"][other] == 2 and r[1]["ivox"][2] == 0
    assert abs(r[1]["s"] - delta / math.sin(abs(eps))) < 1e-9
    assert r[1]["r"][axis] == 0.0                          # snapped to the face
    assert r[0]["u"][axis] * sgn > 0 and r[1]["u"][axis] * sgn < 0
    assert abs(abs(r[1]["u"][axis]) - 9.5e-3) < 1e-3       # theta ~ 11.5 mrad minus the 2 mrad it had
    # step 2: in the neighbour voxel, zero length, back across the same face
    assert r[2]["ivox"][axis] == nb and r[2]["s"] == 0.0 and r[2]["r"][axis] == 0.0
    assert abs(r[2]["E_after"] - r[2]["E_before"]) < 1e-12 and np.allclose(r[2]["u"], r[1]["u"], rtol=0, atol=1e-15)
    # step 3: inside the first voxel again, runs to the z face (9.5 mm away)
    assert r[3]["ivox"][axis] == first and r[3]["ivox"][2] == 0
    assert abs(r[3]["r"][2] - 10.0) < 1e-12 and abs(r[3]["s"] - 9.5) < 1e-3
    assert (r[3]["r"][axis] - 0.0) * sgn < 0               # moved away from the face, into the first voxel
    assert r[4]["ivox"][2] == 1 and r[4]["ivox"][axis] == first
