// vpmc_transport.cuh -- source sampler (S1), range-shifter / aperture module (S2, S3), CT entry and one
// CT voxel step (S4, S5) as device functions.  The production kernels and the trace kernel call exactly
// these functions, so a trace is a faithful record of what the production path does.
#pragma once
#include "vpmc_device.cuh"

namespace vpk {

struct DevTallies {
    double incident, dep_ct, dep_rs, dep_brass, escaped, removed;
    unsigned long long n_stopped_ct, n_stopped_rs, n_stopped_brass, n_nuclear, n_escaped;
    unsigned long long n_steps_ct, n_steps_dev;
};

// per-thread partial tallies
struct Tally {
    double incident = 0, dep_ct = 0, dep_rs = 0, dep_brass = 0, escaped = 0, removed = 0;
    unsigned int n_stopped_ct = 0, n_stopped_rs = 0, n_stopped_brass = 0, n_nuclear = 0, n_escaped = 0;
    unsigned int n_steps_ct = 0, n_steps_dev = 0;
};

struct StepRec {   // == vpmc_step_rec
    unsigned long long hid;
    int step, region, cause;
    int ivox[3];
    float r[3], u[3];
    float E_before, E_after, s;
};

// Tracers record a step with the position converted back to frame coordinates: r = off + (rx, ry, rz).
struct NullTracer {
    __device__ __forceinline__ void put(const Hist &, float, float, float, uint32_t, int, const int *, float, float, float, int) {}
};

struct RecTracer {
    StepRec *recs; int max, n;
    __device__ void put(const Hist &h, float ox, float oy, float oz, uint32_t step, int region, const int *iv,
                        float Eb, float Ea, float s, int cause)
    {
        if (n < max) {
            StepRec &q = recs[n];
            q.hid = ((unsigned long long)h.hid_hi << 32) | h.hid_lo;
            q.step = (int)step; q.region = region; q.cause = cause;
            q.ivox[0] = iv ? iv[0] : -1; q.ivox[1] = iv ? iv[1] : -1; q.ivox[2] = iv ? iv[2] : -1;
            q.r[0] = ox + h.rx; q.r[1] = oy + h.ry; q.r[2] = oz + h.rz; q.u[0] = h.ux; q.u[1] = h.uy; q.u[2] = h.uz;
            q.E_before = Eb; q.E_after = Ea; q.s = s;
        }
        ++n;
    }
};

__device__ __forceinline__ void book_end(Tally &t, int cause, int region, float E_left)
{
    if (cause == ESCAPED) { t.escaped += (double)E_left; t.n_escaped++; }
    else if (cause == NUCLEAR) t.n_nuclear++;
    else if (cause == STOPPED) {
        if (region == REG_CT) t.n_stopped_ct++;
        else if (region == REG_RS) t.n_stopped_rs++;
        else t.n_stopped_brass++;
    }
}

// S1 (C2): sample position, energy and nuclear threshold of history h (hid already set) from spot sp.
// R0 = alpha E_spot^p in fp64 from the host; recomputed on the device only when the source has an energy spread.
__device__ __forceinline__ void sample_source(const DevParams &P, const float4 sp /*x,y,E,sigma*/, double R0,
                                              Hist &h, uint32_t k0, uint32_t k1)
{
    const float4 a = draw4(h, 0u, 1u, k0, k1);
    const float rho = sqrtf(-2.0f * logf(a.x));
    float sn, cs;
    sincospif(2.0f * a.y, &sn, &cs);
    h.rx = fmaf(sp.w, rho * cs, sp.x);
    h.ry = fmaf(sp.w, rho * sn, sp.y);
    h.rz = 0.0f;
    float E0 = sp.z;
    if (P.delta_E != 0.0f) {
        const float zE = sqrtf(-2.0f * logf(a.z)) * cospif(2.0f * a.w);
        E0 = sp.z * fmaf(P.delta_E, zE, 1.0f);
        R0 = (double)P.alpha * pow((double)E0, (double)P.p);
    }
    h.E = E0; h.R = R0;
    const float4 b = draw4(h, 0u, 2u, k0, k1);
    h.tau_star = -logf(b.x);
    h.tau = 0.0f; h.t_rad = 0.0f; h.A_rad = 0.0f; h.step = 0u;
    h.ux = 0.0f; h.uy = 0.0f; h.uz = 1.0f;
}

// vacuum drift over a gap of `gap` mm along w (one step, no RNG); w_to = plane reached (for the record)
template <class Tracer>
__device__ __forceinline__ int drift_gap(Hist &h, float gap, float w_to, Tracer &tr)
{
    if (!(h.uz > 0.0f)) return ESCAPED;
    const float s = fmaxf(__fdiv_rn(gap, h.uz), 0.0f);
    h.rx = fmaf(s, h.ux, h.rx); h.ry = fmaf(s, h.uy, h.ry); h.rz = 0.0f;
    tr.put(h, 0.0f, 0.0f, w_to, h.step, REG_VAC, nullptr, h.E, h.E, s, CONT);
    h.step += 1u;
    return CONT;
}

__device__ __forceinline__ bool aperture_open(const DevBeam &b, float x, float y)
{
    const float fx = floorf(__fdiv_rn(x - b.ap_u0, b.ap_du)), fy = floorf(__fdiv_rn(y - b.ap_v0, b.ap_dv));
    if (!(fx >= 0.0f && fx < (float)b.ap_nx && fy >= 0.0f && fy < (float)b.ap_ny)) return false;
    const int ix = (int)fx, iy = (int)fy;
    const uint32_t wv = __ldg(b.ap_bits + (size_t)iy * b.ap_row_words + (ix >> 5));
    return (wv >> (ix & 31)) & 1u;
}

// S2 + S3 (C3): start plane -> range shifter -> aperture, in the beam frame with rz = local depth in the device.
// Returns CONT when the history left the last device alive (or there is none), else the terminating cause;
// w_now = beam-frame w of the plane the history stands on.
template <class Tracer>
__device__ int beamline(const DevParams &P, const DevBeam &b, Hist &h, Tally &t, Tracer &tr, uint32_t k0, uint32_t k1,
                        float &w_now)
{
    StepOut o;
    w_now = b.w_start;
    if (b.has_rs) {
        if (drift_gap(h, b.w_rs_in - w_now, b.w_rs_in, tr) != CONT) goto escaped;
        const Medium m = { P.rs_rsp, P.rs_rho, P.rs_inv_X0, P.rs_za_rho };
        const float T = b.w_rs_out - b.w_rs_in;
        w_now = b.w_rs_in;
        for (;;) {
            if (!(h.uz > 0.0f)) goto escaped;
            float d = P.s_rs; const float dist = __fdiv_rn(T - h.rz, h.uz); int ex = 0;
            if (dist <= d) { d = dist; ex = 1; }
            d = fmaxf(d, 0.0f);
            const float Eb = h.E; const uint32_t st = h.step;
            const int cause = material_step(P, h, m, d, k0, k1, o);
            t.dep_rs += (double)o.dep; t.removed += (double)o.removed;
            const bool out = (cause == CONT) && o.on_d && ex;
            if (out) h.rz = T;
            tr.put(h, 0.0f, 0.0f, b.w_rs_in, st, REG_RS, nullptr, Eb, h.E, o.s, cause);
            if (cause != CONT) { book_end(t, cause, REG_RS, 0.0f); return cause; }
            if (out) break;
        }
        w_now = b.w_rs_out;
    }
    if (b.has_ap) {
        if (drift_gap(h, b.w_ap_in - w_now, b.w_ap_in, tr) != CONT) goto escaped;
        const Medium m = { P.brass_rsp, P.brass_rho, P.brass_inv_X0, P.brass_za_rho };
        const float T = b.w_ap_out - b.w_ap_in;
        w_now = b.w_ap_in;
        for (;;) {
            if (!(h.uz > 0.0f)) goto escaped;
            float d = P.s_ap; const float dist = __fdiv_rn(T - h.rz, h.uz); int ex = 0;
            if (dist <= d) { d = dist; ex = 1; }
            d = fmaxf(d, 0.0f);
            if (aperture_open(b, h.rx, h.ry)) {     // transported with the previous velocity and direction
                h.rx = fmaf(d, h.ux, h.rx); h.ry = fmaf(d, h.uy, h.ry); h.rz = ex ? T : fmaf(d, h.uz, h.rz);
                tr.put(h, 0.0f, 0.0f, b.w_ap_in, h.step, REG_AP_OPEN, nullptr, h.E, h.E, d, CONT);
                h.step += 1u;
                if (ex) break;
                continue;
            }
            const float Eb = h.E; const uint32_t st = h.step;
            const int cause = material_step(P, h, m, d, k0, k1, o);
            t.dep_brass += (double)o.dep; t.removed += (double)o.removed;
            const bool out = (cause == CONT) && o.on_d && ex;
            if (out) h.rz = T;
            tr.put(h, 0.0f, 0.0f, b.w_ap_in, st, REG_AP_BRASS, nullptr, Eb, h.E, o.s, cause);
            if (cause != CONT) { book_end(t, cause, REG_AP_BRASS, 0.0f); return cause; }
            if (out) break;
        }
        w_now = b.w_ap_out;
    }
    h.rz = 0.0f;
    return CONT;
escaped:
    tr.put(h, 0.0f, 0.0f, w_now, h.step, REG_VAC, nullptr, h.E, h.E, 0.0f, ESCAPED);
    book_end(t, ESCAPED, REG_VAC, h.E);
    return ESCAPED;
}

// Beam frame -> CT frame (setup shift moves the patient), ray-box entry, entry voxel (C3).  On return the
// position variables are LOCAL offsets inside voxel iv.
template <class Tracer>
__device__ int enter_ct(const DevGrid &G, const DevBeam &b, const float shift[3], float w_now, Hist &h, int iv[3],
                        Tally &t, Tracer &tr)
{
    float r[3], u[3];
    {
        const float x = h.rx, y = h.ry, z = w_now, a = h.ux, c = h.uy, e = h.uz;
        r[0] = (b.iso[0] - shift[0]) + (b.rot[0] * x + b.rot[1] * y + b.rot[2] * z);
        r[1] = (b.iso[1] - shift[1]) + (b.rot[3] * x + b.rot[4] * y + b.rot[5] * z);
        r[2] = (b.iso[2] - shift[2]) + (b.rot[6] * x + b.rot[7] * y + b.rot[8] * z);
        u[0] = b.rot[0] * a + b.rot[1] * c + b.rot[2] * e;
        u[1] = b.rot[3] * a + b.rot[4] * c + b.rot[5] * e;
        u[2] = b.rot[6] * a + b.rot[7] * c + b.rot[8] * e;
        h.ux = u[0]; h.uy = u[1]; h.uz = u[2];
    }
    const float lo[3] = { G.ox, G.oy, G.oz };
    const float hh[3] = { G.hx, G.hy, G.hz };
    const int n[3] = { G.nx, G.ny, G.nz };
    float t_in = 0.0f, t_out = __int_as_float(0x7f800000); int ax = -1; bool miss = false;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const float hi = lo[a] + (float)n[a] * hh[a];
        if (u[a] == 0.0f) { if (r[a] < lo[a] || r[a] >= hi) miss = true; continue; }
        const float t1 = __fdiv_rn(lo[a] - r[a], u[a]), t2 = __fdiv_rn(hi - r[a], u[a]);
        const float tn = fminf(t1, t2), tf = fmaxf(t1, t2);
        if (tn > t_in) { t_in = tn; ax = a; }
        t_out = fminf(t_out, tf);
    }
    if (miss || !(t_in < t_out)) {
        h.rx = r[0]; h.ry = r[1]; h.rz = r[2];
        tr.put(h, 0.0f, 0.0f, 0.0f, h.step, REG_VAC, nullptr, h.E, h.E, 0.0f, ESCAPED);
        book_end(t, ESCAPED, REG_VAC, h.E);
        return ESCAPED;
    }
    float l[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const float q = fmaf(t_in, u[a], r[a]);
        if (a == ax) {
            if (u[a] > 0.0f) { iv[a] = 0; l[a] = 0.0f; } else { iv[a] = n[a] - 1; l[a] = hh[a]; }
        } else {
            float f = floorf(__fdiv_rn(q - lo[a], hh[a]));
            f = fminf(fmaxf(f, 0.0f), (float)(n[a] - 1));
            iv[a] = (int)f;
            l[a] = fminf(fmaxf(q - fmaf(f, hh[a], lo[a]), 0.0f), hh[a]);
        }
    }
    h.rx = l[0]; h.ry = l[1]; h.rz = l[2];
    tr.put(h, fmaf((float)iv[0], G.hx, G.ox), fmaf((float)iv[1], G.hy, G.oy), fmaf((float)iv[2], G.hz, G.oz),
           h.step, REG_VAC, nullptr, h.E, h.E, t_in, CONT);
    h.step += 1u;
    return CONT;
}

// S4: distance to the nearest face of the current voxel from the local offset, ties to the lowest axis
__device__ __forceinline__ float face_distance(const DevGrid &G, const Hist &h, int &ax)
{
    const float inf = __int_as_float(0x7f800000);
    float dx = inf, dy = inf, dz = inf;
    if (h.ux > 0.0f) dx = __fdividef(G.hx - h.rx, h.ux); else if (h.ux < 0.0f) dx = __fdividef(-h.rx, h.ux);
    if (h.uy > 0.0f) dy = __fdividef(G.hy - h.ry, h.uy); else if (h.uy < 0.0f) dy = __fdividef(-h.ry, h.uy);
    if (h.uz > 0.0f) dz = __fdividef(G.hz - h.rz, h.uz); else if (h.uz < 0.0f) dz = __fdividef(-h.rz, h.uz);
    float d = dx; ax = 0;
    if (dy < d) { d = dy; ax = 1; }
    if (dz < d) { d = dz; ax = 2; }
    return fmaxf(d, 0.0f);
}

// C4-9: the step ended on a voxel face: advance that index, snap that local coordinate.  `up` = direction sign
// on that axis BEFORE the scattering of this step.  Returns true if the history left the grid.
__device__ __forceinline__ bool cross_face(const DevGrid &G, Hist &h, int &ix, int &iy, int &iz, int ax, bool up)
{
    if (ax == 0) {
        if (up) { ix += 1; h.rx = 0.0f; } else { ix -= 1; h.rx = G.hx; }
        return ix < 0 || ix >= G.nx;
    } else if (ax == 1) {
        if (up) { iy += 1; h.ry = 0.0f; } else { iy -= 1; h.ry = G.hy; }
        return iy < 0 || iy >= G.ny;
    } else {
        if (up) { iz += 1; h.rz = 0.0f; } else { iz -= 1; h.rz = G.hz; }
        return iz < 0 || iz >= G.nz;
    }
}

}  // namespace vpk
