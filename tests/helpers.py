"""Shared test helpers: workload dict -> oracle Problem, and small utilities."""
import numpy as np

from oracle import vpmc_oracle as orc


def oracle_problem(wl: dict, params=None, f32_params=True) -> orc.Problem:
    p = params if params is not None else orc.default_params()
    if f32_params:
        p = orc.params_as_f32(p)
    return orc.Problem(ct=wl["ct"], calib=wl["calib"], beams=wl["beams"], params=p)


def grid(wl, flat):
    n = wl["ct"]["n"]
    return np.asarray(flat).reshape(n[2], n[1], n[0])


def read_golden(name):
    """Whitespace-separated rows, '#' comments."""
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", name)
    rows = []
    with open(path) as f:
        for line in f:
            line = line.split("#", 1)[0].strip()
            if line:
                rows.append(line.split())
    return rows


# ---- the single-threaded oracle over all host cores: independent processes on disjoint history-id ranges (legal because
# streams are keyed by history id); used by the full-size window parity tests

def _window_worker(args):
    fn, kw, N, seed, lo, hi, sc, hps, g, want_digests = args
    from oracle import vpmc_oracle as O
    from paper_2307_01416_b200 import workloads
    w = getattr(workloads, fn)(**kw)
    pb = oracle_problem(w)
    s = None if sc is None else O.scenario(sc[0], float(np.float32(sc[1])))
    if g is None:
        e, t = O.dose_edep(pb, N, seed, s, hid_begin=lo, hid_end=hi)
    else:
        e, t = O.influence_edep(pb, g, hps, seed, s, i_begin=lo, i_end=hi)
    nz = np.flatnonzero(e)
    dig = O.digests(pb, N, seed, lo, hi - lo, s) if want_digests else None
    return nz.astype(np.int64), e[nz], t.as_dict(), dig


def _merge(res, nvox):
    e = np.zeros(nvox, dtype=np.float64)
    tal = None
    for idx, val, t, _ in res:
        e[idx] += val
        tal = dict(t) if tal is None else {k: tal[k] + t[k] for k in tal}
    return e, tal


def n_cores():
    import os
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def oracle_window_parallel(fn, kw, nvox, N, seed, lo, hi, sc=None, digests=False):
    """E_dep (fp64, MeV) and tallies (dict) of history ids [lo, hi) of the N-history dose run of workload fn(**kw);
    with digests=True also the per-history digests (oracle DIGEST_DTYPE, in id order)."""
    import multiprocessing as mp
    k = max(1, min(n_cores(), (hi - lo) // 2000))
    cuts = [lo + (hi - lo) * i // k for i in range(k + 1)]
    jobs = [(fn, kw, N, seed, cuts[i], cuts[i + 1], sc, 0, None, digests) for i in range(k)]
    with mp.get_context("spawn").Pool(k) as pool:
        res = pool.map(_window_worker, jobs)
    e, tal = _merge(res, nvox)
    if digests:
        return e, tal, np.concatenate([r[3] for r in res])
    return e, tal


def oracle_columns_parallel(fn, kw, nvox, spots, hps, seed, sc=None):
    """E_dep per influence column (list of fp64 arrays) of the given global spots, hist_per_spot = hps."""
    import multiprocessing as mp
    k = n_cores()
    per = max(1, -(-k // max(len(spots), 1)))              # slices per column so that all cores are busy
    jobs = []
    for g in spots:
        cuts = [hps * i // per for i in range(per + 1)]
        jobs += [(fn, kw, 0, seed, cuts[i], cuts[i + 1], sc, hps, int(g), False) for i in range(per)]
    with mp.get_context("spawn").Pool(min(k, len(jobs))) as pool:
        res = pool.map(_window_worker, jobs)
    return [_merge(res[j * per:(j + 1) * per], nvox)[0] for j in range(len(spots))]


def polygon_edge_distance(poly, x, y):
    """Euclidean distance of (x, y) to the boundary of the closed polygon poly [n, 2] (numpy, fp64)."""
    p = np.asarray(poly, dtype=np.float64).reshape(-1, 2)
    q = np.roll(p, -1, axis=0)
    e = q - p
    l2 = np.maximum((e * e).sum(axis=1), 1e-300)
    t = np.clip(((np.array([x, y]) - p) * e).sum(axis=1) / l2, 0.0, 1.0)
    d = p + t[:, None] * e - np.array([x, y])
    return float(np.sqrt((d * d).sum(axis=1).min()))


def deciding_gap(O, w, P, kind, beam, E, E0, r, u, ivox, tau_after, tau_star, extent):
    """the smallest relative gap of the discrete decisions of one step (kind 'ct' | 'rs' | 'ap'),
    evaluated in the ORACLE's pre-step state: how far, relative to the fixed scales (grid extent, R0, 1), the state is
    from the point where a decision flips -- which face is reached first, face or range limit, exit-plane test, stop
    test, nuclear threshold, sign of a direction cosine, pixel edge of the opening bitmap.  Path-length gaps are
    converted to the position change that closes them (times the direction cosine of that axis)."""
    r, u = np.asarray(r, dtype=np.float64), np.asarray(u, dtype=np.float64)
    R = P.alpha * E ** P.p
    R0 = P.alpha * E0 ** P.p
    gaps = [abs(R - P.R_cut) / R0, abs(tau_after - tau_star)]
    b = w["beams"][beam]
    if kind == "ct":
        ct = w["ct"]
        n, h, o = np.array(ct["n"]), np.array(ct["h"], dtype=np.float64), np.array(ct["origin"], dtype=np.float64)
        iv = np.asarray(ivox, dtype=np.int64)
        d = []
        for a in range(3):
            if u[a] > 0: d.append((max((o[a] + (iv[a] + 1) * h[a] - r[a]) / u[a], 0.0), abs(u[a])))
            elif u[a] < 0: d.append((max((o[a] + iv[a] * h[a] - r[a]) / u[a], 0.0), abs(u[a])))
            gaps.append(abs(u[a]))
        d.sort()
        if len(d) > 1: gaps.append((d[1][0] - d[0][0]) * min(d[0][1], d[1][1]) / extent)
        hu = float(np.asarray(ct["hu"]).reshape(n[2], n[1], n[0])[iv[2], iv[1], iv[0]])
        rsp = O.calib_eval(w["calib"], hu)[0]
        lim = max(P.f_R * R, P.R_cut) / rsp
        gaps.append(min(abs(d[0][0] - lim) * d[0][1] / extent, abs(d[0][0] - lim) * rsp / P.f_R / R0))
    elif kind in ("rs", "ap"):
        rs = kind == "rs"
        w_out = -float(b["rs_face"] if rs else b["aperture"]["face"])
        d0 = P.s_rs if rs else P.s_ap
        dist = (w_out - r[2]) / u[2] if u[2] > 0 else 0.0
        gaps += [abs(dist - d0) * abs(u[2]) / extent, abs(u[2])]
        rsp = P.rs_rsp if rs else P.brass_rsp
        gaps.append(abs(min(d0, dist) - max(P.f_R * R, P.R_cut) / rsp) * rsp / P.f_R / R0)
        if not rs and b["aperture"].get("polygon") is not None:      # polygon opening: distance to the nearest edge
            gaps.append(polygon_edge_distance(b["aperture"]["polygon"], r[0], r[1]) / extent)
        elif not rs:
            ap = b["aperture"]
            for x, x0, dx in ((r[0], float(ap["u0"]), float(ap["du"])), (r[1], float(ap["v0"]), float(ap["dv"]))):
                f = (x - x0) / dx
                gaps.append(abs(f - round(f)) * dx / extent)
    return min(gaps)
