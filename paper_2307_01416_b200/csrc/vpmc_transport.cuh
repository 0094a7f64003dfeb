// vpmc_transport.cuh -- the two step functions of the hot path: beam_step() = one iteration of a history in the beam
// line (S1 source, S2 range shifter, S3 aperture module) and ct_step() = one voxel step (S4, S5, scoring hook S6/S7),
// plus the CT entry.  The production kernels and the trace kernel call exactly these functions, so a trace is a
// faithful record of what the production path does.
//
// Control structure ("identical control logic"): a warp only ever holds histories of ONE stage -- beam line or
// CT -- so its lanes run the same code.  Inside the beam line the range shifter and the brass are the same slab step
// with different constants; only the drift through the aperture opening differs, and it is cheap.
#pragma once
#include "vpmc_device.cuh"

namespace vpk {

struct DevTallies {
    double incident, dep_ct, dep_rs, dep_brass, escaped, removed;
    unsigned long long n_stopped_ct, n_stopped_rs, n_stopped_brass, n_nuclear, n_escaped;
    unsigned long long n_steps_ct, n_steps_dev, n_steps_slab;
};
enum : int { TD_INCIDENT = 0, TD_DEP_CT, TD_DEP_RS, TD_DEP_BRASS, TD_ESCAPED, TD_REMOVED, TD_N };
enum : int { TC_STOP_CT = 0, TC_STOP_RS, TC_STOP_BRASS, TC_NUCLEAR, TC_ESCAPED, TC_STEPS_CT, TC_STEPS_DEV, TC_STEPS_SLAB, TC_N };

// per-warp partial tallies in shared memory (fp64 sums; flushed to DevTallies once per warp at kernel end)
struct WarpTally { double d[TD_N]; unsigned int c[TC_N]; };

struct SmemSink {
    WarpTally *w;
    __device__ __forceinline__ void add_d(int k, float v) const { if (v != 0.0f) atomicAdd(&w->d[k], (double)v); }
    __device__ __forceinline__ void add_c(int k, unsigned n) const { if (n) atomicAdd(&w->c[k], n); }
};
struct NullSink {
    __device__ __forceinline__ void add_d(int, float) const {}
    __device__ __forceinline__ void add_c(int, unsigned) const {}
};

struct StepRec {   // == vpmc_step_rec
    unsigned long long hid;
    int step, region, cause;
    int ivox[3];
    float r[3], u[3];
    float E_before, E_after, s;
    float dep; int pad_;         // energy deposited in the step's cell (CT voxel, range shifter or brass tally), MeV
};

struct NullTracer {
    static constexpr bool on = false;
    __device__ __forceinline__ void put(const Hist &, float, float, float, uint32_t, int, const int *, float, float, float, int, float = 0.0f) {}
};

struct RecTracer {
    static constexpr bool on = true;
    StepRec *recs; int max, n;
    __device__ void put(const Hist &h, float x, float y, float z, uint32_t step, int region, const int *iv,
                        float Eb, float Ea, float s, int cause, float dep = 0.0f)
    {
        if (n < max) {
            StepRec &q = recs[n];
            q.hid = ((unsigned long long)h.hid_hi << 32) | h.hid_lo;
            q.step = (int)step; q.region = region; q.cause = cause;
            q.ivox[0] = iv ? iv[0] : -1; q.ivox[1] = iv ? iv[1] : -1; q.ivox[2] = iv ? iv[2] : -1;
            q.r[0] = x; q.r[1] = y; q.r[2] = z;
            q.u[0] = h.ux + h.lx; q.u[1] = h.uy + h.ly; q.u[2] = h.uz + h.lz;
            q.E_before = Eb; q.E_after = Ea; q.s = s; q.dep = dep; q.pad_ = 0;
        }
        ++n;
    }
};

// Per-history digest instead of step records (vpmc_digest, test-only): number of records, FNV-1a hash of the discrete
// trace (region, cause, voxel indices of every record), state after the last record and the energy deposited in the CT.
struct Digest {   // == vpmc_digest
    unsigned long long hid, hash;
    int n_rec, cause;
    float r[3];
    float E_last, dep_ct;
    int pad_;
};
struct DigestTracer {
    static constexpr bool on = true;
    Digest d; int n;
    __device__ void start(unsigned long long hid) { d.hid = hid; d.hash = 1469598103934665603ull; d.n_rec = 0; d.cause = 0; d.r[0] = d.r[1] = d.r[2] = 0.0f; d.E_last = 0.0f; d.dep_ct = 0.0f; d.pad_ = 0; n = 0; }
    __device__ void mix(unsigned int v) { d.hash = (d.hash ^ (unsigned long long)v) * 1099511628211ull; }
    __device__ void put(const Hist &, float x, float y, float z, uint32_t, int region, const int *iv, float, float Ea, float, int cause, float = 0.0f)
    {
        mix((unsigned)region); mix((unsigned)cause);
        mix((unsigned)(iv ? iv[0] : -1)); mix((unsigned)(iv ? iv[1] : -1)); mix((unsigned)(iv ? iv[2] : -1));
        d.n_rec += 1; d.cause = cause; d.r[0] = x; d.r[1] = y; d.r[2] = z; d.E_last = Ea;
        ++n;
    }
};

// everything a step needs besides the history itself (kernel arguments -> constant bank)
struct Ctx {
    DevParams P;
    DevGrid G;
    const DevBeam *beams;
    const short *hu;
    float rsp_scale, inv_rsp_scale;
    float shift[3];
    PhiloxKey K;
};

// S1 (C2): sample position, energy and nuclear threshold of history h (hid already set) from spot sp.
// R0 = alpha E_spot^p in fp64 from the host; recomputed on the device only when the source has an energy spread.
__device__ __forceinline__ void sample_source(const DevParams &P, const DevBeam &b, int beam, const float4 sp /*x,y,E,sigma*/,
                                              double R0, Hist &h, const PhiloxKey &K)
{
    const float4 a = draw4(h, 0u, 1u, K);
    const float rho = sqrtf(-2.0f * logf(a.x));
    float sn, cs;
    sincospif(2.0f * a.y, &sn, &cs);
    set_beam_x(h, fma((double)sp.w, (double)(rho * cs), (double)sp.x));
    set_beam_y(h, fma((double)sp.w, (double)(rho * sn), (double)sp.y));
    h.rx = 0.0f; h.ry = 0.0f; h.rz = 0.0f;
    float E0 = sp.z;
    if (P.delta_E != 0.0f) {
        const float zE = sqrtf(-2.0f * logf(a.z)) * cospif(2.0f * a.w);
        const float dl = P.delta_E * zE;
        E0 = sp.z * (1.0f + dl);
        R0 = fma(R0, (double)expm1f(P.p * log1pf(dl)), R0);      // alpha (E (1 + dl))^p = R0 (1 + dl)^p
    }
    h.E = E0; h.R = R0;
    const float4 c = draw4(h, 0u, 2u, K);
    h.tau_star = -logf(c.x);
    h.tau = 0.0f; h.t_rad = 0.0f; h.f_rad = 1.0f; h.step = 0u;
    h.ux = 0.0f; h.uy = 0.0f; h.uz = 1.0f; h.lx = 0.0f; h.ly = 0.0f; h.lz = 0.0f;
    h.region = (b.has_rs ? REG_TO_RS : (b.has_ap ? REG_TO_AP : REG_TO_CT)) | (beam << 8);
}

// vacuum drift over a gap of `gap` mm along w (one step, no RNG); w_to = plane reached (for the record)
template <class Tracer>
__device__ __forceinline__ int drift_gap(Hist &h, float gap, float w_to, Tracer &tr)
{
    if (!(h.uz > 0.0f)) return ESCAPED;
    const double uz = (double)h.uz + (double)h.lz;
    const double s = fmax((double)gap / uz, 0.0);
    const double x = fma(s, (double)h.ux + (double)h.lx, beam_x(h)), y = fma(s, (double)h.uy + (double)h.ly, beam_y(h));
    set_beam_x(h, x); set_beam_y(h, y);
    h.rz = 0.0f;
    if (Tracer::on) tr.put(h, (float)x, (float)y, w_to, h.step, REG_VAC, nullptr, h.E, h.E, (float)s, CONT);
    h.step += 1u;
    return CONT;
}

// the medium under the current (u, v): bit of the opening bitmap; outside the bitmap = brass.  The pixel index
// is taken in fp32 from the high part of the position: an error of ~4e-6 mm only matters within that distance of the
// opening's edge.  (ix, iy) are returned for the safe-distance lookup.
__device__ __forceinline__ bool aperture_open(const DevBeam *b, float x, float y, int &ix, int &iy)
{
    const float fx = floorf((x - __ldg(&b->ap_u0)) * __ldg(&b->ap_inv_du)), fy = floorf((y - __ldg(&b->ap_v0)) * __ldg(&b->ap_inv_dv));
    const int nx = __ldg(&b->ap_nx), ny = __ldg(&b->ap_ny);
    if (!(fx >= 0.0f && fx < (float)nx && fy >= 0.0f && fy < (float)ny)) { ix = iy = -1; return false; }
    ix = (int)fx; iy = (int)fy;
    const uint32_t wv = __ldg(b->ap_bits + (size_t)iy * __ldg(&b->ap_row_words) + (ix >> 5));
    return (wv >> (ix & 31)) & 1u;
}

// S:8f-2 (ref. 67): crossing-number test of (x, y) against the closed polygon, edge k = vertex k -> vertex k + 1 --
// an edge counts when its end points lie on different sides of the line through y and it meets that line right of x -- and,
// in the same pass, the squared distance to the nearest edge.  Kept out of line: it is called once or twice per history and
// must not cost the step loops their registers.
__device__ __noinline__ bool polygon_query(const float2 *__restrict__ poly, int n, float x, float y, float &dist2)
{
    bool inside = false;
    float d2 = 1e30f;
    float2 a = __ldg(poly + n - 1);
    for (int k = 0; k < n; ++k) {
        const float2 b = __ldg(poly + k);
        const float ex = b.x - a.x, ey = b.y - a.y, px = x - a.x, py = y - a.y;
        if ((a.y > y) != (b.y > y)) {
            const float xi = a.x + __fdiv_rn(py * ex, ey);
            if (x < xi) inside = !inside;
        }
        const float l2 = fmaf(ex, ex, ey * ey);
        const float t = (l2 > 0.0f) ? fminf(fmaxf(__fdiv_rn(fmaf(px, ex, py * ey), l2), 0.0f), 1.0f) : 0.0f;
        const float dx = fmaf(-t, ex, px), dy = fmaf(-t, ey, py);
        d2 = fminf(d2, fmaf(dx, dx, dy * dy));
        a = b;
    }
    dist2 = d2;
    return inside;
}

// The same test for a point of grid row `row`, over the edges that can matter there: the crossing count over the row's own
// edge list (an edge outside it has both end points on one side of the ray's line: the full loop would skip it too, so the
// answer is the full loop's), the distance over the lists of the rows row - 1 .. row + 1 -- any other edge is at least one
// cell away, so the distance is capped at one cell.
__device__ __noinline__ bool polygon_query_row(const DevBeam *bp, int row, float x, float y, float &dist2)
{
    const float2 *__restrict__ poly = bp->ap_poly;
    const int *__restrict__ rp = bp->ap_prow_ptr, *__restrict__ ed = bp->ap_pedges;
    const int n = __ldg(&bp->ap_n_poly), ny = __ldg(&bp->ap_pg_ny);
    const float cell = __frcp_rn(__ldg(&bp->ap_pg_inv_cell));
    bool inside = false;
    float d2 = cell * cell;
    for (int r = max(row - 1, 0); r <= min(row + 1, ny - 1); ++r)
        for (int i = __ldg(rp + r); i < __ldg(rp + r + 1); ++i) {
            const int k = __ldg(ed + i);
            const float2 a = __ldg(poly + k), b = __ldg(poly + (k + 1 == n ? 0 : k + 1));
            const float ex = b.x - a.x, ey = b.y - a.y, px = x - a.x, py = y - a.y;
            if (r == row && (a.y > y) != (b.y > y)) {
                const float xi = a.x + __fdiv_rn(py * ex, ey);
                if (x < xi) inside = !inside;
            }
            const float l2 = fmaf(ex, ex, ey * ey);
            const float t = (l2 > 0.0f) ? fminf(fmaxf(__fdividef(fmaf(px, ex, py * ey), l2), 0.0f), 1.0f) : 0.0f;
            const float dx = fmaf(-t, ex, px), dy = fmaf(-t, ey, py);
            d2 = fminf(d2, fmaf(dx, dx, dy * dy));
        }
    dist2 = d2;
    return inside;
}

// The medium under (x, y) of either kind of opening, with the lateral travel (L-infinity norm, mm, per axis) over which the
// answer is KNOWN not to change -- 0 when nothing is known (the per-step test of P:L87 is kept in outcome,
// tests whose answer is known are not executed).
__device__ __forceinline__ bool aperture_query(const DevBeam *bp, float x, float y, float &safe_u, float &safe_v)
{
    if (__ldg(&bp->ap_n_poly) > 0) {
        const float gx = (x - __ldg(&bp->ap_pg_x0)) * __ldg(&bp->ap_pg_inv_cell), gy = (y - __ldg(&bp->ap_pg_y0)) * __ldg(&bp->ap_pg_inv_cell);
        const int nx = __ldg(&bp->ap_pg_nx), ny = __ldg(&bp->ap_pg_ny);
        if (!(gx >= 0.0f && gx < (float)nx && gy >= 0.0f && gy < (float)ny)) {
            // outside the grid (which covers the polygon's bounding box): brass at least up to the grid's rectangle
            const float cell = __frcp_rn(__ldg(&bp->ap_pg_inv_cell));
            const float d = fmaxf(fmaxf(-gx, gx - (float)nx), fmaxf(-gy, gy - (float)ny)) * cell;
            safe_u = safe_v = 0.99f * fmaxf(d, 0.0f);
            return false;
        }
        const float cv = __ldg(bp->ap_pgrid + (size_t)(int)gy * nx + (int)gx);
        if (cv != 0.0f) { safe_u = safe_v = fabsf(cv); return cv > 0.0f; }
        float d2;
        const bool in = polygon_query_row(bp, (int)gy, x, y, d2);
        safe_u = safe_v = 0.7f * sqrt_fast(d2);          // Euclidean radius d -> L-infinity radius d / sqrt(2), rounded down
        return in;
    }
    int ix, iy;
    const bool open = aperture_open(bp, x, y, ix, iy);
    if (ix < 0) {        // outside the bitmap: brass up to its rectangle
        const float u0 = __ldg(&bp->ap_u0), v0 = __ldg(&bp->ap_v0);
        const float u1 = u0 + (float)__ldg(&bp->ap_nx) * __frcp_rn(__ldg(&bp->ap_inv_du)), v1 = v0 + (float)__ldg(&bp->ap_ny) * __frcp_rn(__ldg(&bp->ap_inv_dv));
        safe_u = safe_v = 0.99f * fmaxf(fmaxf(u0 - x, x - u1), fmaxf(v0 - y, y - v1));
        return false;
    }
    // k tiles to the nearest tile of the other kind -> (k - 1) tiles of lateral travel are safe
    const unsigned char *map = open ? bp->ap_dist : bp->ap_dist_open;
    const int k = (int)__ldg(map + (size_t)(iy >> kApTileShift) * __ldg(&bp->ap_ntx) + (ix >> kApTileShift));
    const float safe = (k >= 2) ? 0.99f * (float)(k - 1) : 0.0f;
    safe_u = safe * __ldg(&bp->ap_tile_u); safe_v = safe * __ldg(&bp->ap_tile_v);
    return open;
}

// Beam frame -> CT frame (setup shift moves the patient), ray-box entry, entry voxel (C3).  Done in fp64: it runs
// once per history and fixes the entry point that every later face crossing inherits.  On return the geometry
// slots hold ix, iy, iz, v and rx, ry, rz are LOCAL offsets inside that voxel.
template <class Tracer>
__device__ __forceinline__ int enter_ct(const Ctx &c, const DevBeam &b, float w_now, Hist &h, Tracer &tr)
{
    const DevGrid &G = c.G;
    double r[3], u[3];
    {
        const double x = beam_x(h), y = beam_y(h), z = (double)w_now;
        const double a = (double)h.ux + (double)h.lx, q = (double)h.uy + (double)h.ly, e = (double)h.uz + (double)h.lz;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            r[k] = ((double)b.iso[k] - (double)c.shift[k]) + (double)b.rot[3 * k] * x + (double)b.rot[3 * k + 1] * y + (double)b.rot[3 * k + 2] * z;
            u[k] = (double)b.rot[3 * k] * a + (double)b.rot[3 * k + 1] * q + (double)b.rot[3 * k + 2] * e;
        }
    }
    h.ux = (float)u[0]; h.uy = (float)u[1]; h.uz = (float)u[2];
    h.lx = (float)(u[0] - (double)h.ux); h.ly = (float)(u[1] - (double)h.uy); h.lz = (float)(u[2] - (double)h.uz);
    const double lo[3] = { (double)G.ox, (double)G.oy, (double)G.oz };
    const double hh[3] = { (double)G.hx, (double)G.hy, (double)G.hz };
    const int n[3] = { G.nx, G.ny, G.nz };
    double t_in = 0.0, t_out = __longlong_as_double(0x7ff0000000000000LL); int ax = -1; bool miss = false;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double hi = lo[a] + (double)n[a] * hh[a];
        if (u[a] == 0.0) { if (r[a] < lo[a] || r[a] >= hi) miss = true; continue; }
        const double t1 = (lo[a] - r[a]) / u[a], t2 = (hi - r[a]) / u[a];
        const double tn = fmin(t1, t2), tf = fmax(t1, t2);
        if (tn > t_in) { t_in = tn; ax = a; }
        t_out = fmin(t_out, tf);
    }
    if (miss || !(t_in < t_out)) {
        if (Tracer::on) tr.put(h, (float)r[0], (float)r[1], (float)r[2], h.step, REG_VAC, nullptr, h.E, h.E, 0.0f, ESCAPED);
        return ESCAPED;
    }
    int iv[3]; float l[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double q = fma(t_in, u[a], r[a]);
        if (a == ax) {
            if (u[a] > 0.0) { iv[a] = 0; l[a] = 0.0f; } else { iv[a] = n[a] - 1; l[a] = (float)hh[a]; }
        } else {
            double f = floor((q - lo[a]) / hh[a]);
            f = fmin(fmax(f, 0.0), (double)(n[a] - 1));
            iv[a] = (int)f;
            l[a] = (float)fmin(fmax(q - fma(f, hh[a], lo[a]), 0.0), hh[a]);
        }
    }
    h.rx = l[0]; h.ry = l[1]; h.rz = l[2];
    h.g0 = (uint32_t)iv[0]; h.g1 = (uint32_t)iv[1]; h.g2 = (uint32_t)iv[2];
    h.g3 = (uint32_t)(iv[0] + G.nx * (iv[1] + G.ny * iv[2]));
    if (Tracer::on) tr.put(h, fmaf((float)iv[0], G.hx, G.ox) + l[0], fmaf((float)iv[1], G.hy, G.oy) + l[1], fmaf((float)iv[2], G.hz, G.oz) + l[2],
                           h.step, REG_VAC, nullptr, h.E, h.E, (float)t_in, CONT);
    h.step += 1u;
    return CONT;
}

// S4: distance to the nearest face of the current voxel from the local offset.  The nearest axis is found by
// cross-multiplication (dist_a |u_b| < dist_b |u_a|), so only ONE reciprocal goes through the MUFU pipe; ties go to the
// lowest axis.  `up` = the history moves towards +axis on that axis during the step.
__device__ __forceinline__ float face_distance(const DevGrid &G, const Hist &h, int &ax, bool &up)
{
    float nx = (h.ux > 0.0f) ? G.hx - h.rx : h.rx, ax_ = fabsf(h.ux);
    float ny = (h.uy > 0.0f) ? G.hy - h.ry : h.ry, ay_ = fabsf(h.uy);
    float nz = (h.uz > 0.0f) ? G.hz - h.rz : h.rz, az_ = fabsf(h.uz);
    if (ax_ == 0.0f) { nx = 1e30f; ax_ = 1.0f; }
    if (ay_ == 0.0f) { ny = 1e30f; ay_ = 1.0f; }
    if (az_ == 0.0f) { nz = 1e30f; az_ = 1.0f; }
    float n = nx, a = ax_; ax = 0; up = h.ux > 0.0f;
    if (ny * a < n * ay_) { n = ny; a = ay_; ax = 1; up = h.uy > 0.0f; }
    if (nz * a < n * az_) { n = nz; a = az_; ax = 2; up = h.uz > 0.0f; }
    return fmaxf(__fdividef(n, a), 0.0f);
}

// C4-9: the step ended on a voxel face: advance that index, snap that local coordinate.  `up` = direction sign
// on that axis BEFORE the scattering of this step.  Returns true if the history left the grid.
__device__ __forceinline__ bool cross_face(const DevGrid &G, Hist &h, int ax, bool up)
{
    // a three-way branch on purpose: the select-only version measured twice the instructions (profiles/r1_README.md)
    if (ax == 0) {
        if (up) { h.g0 += 1u; h.g3 += 1u; h.rx = 0.0f; } else { h.g0 -= 1u; h.g3 -= 1u; h.rx = G.hx; }
        return h.g0 >= (uint32_t)G.nx;
    } else if (ax == 1) {
        if (up) { h.g1 += 1u; h.g3 += (uint32_t)G.nx; h.ry = 0.0f; } else { h.g1 -= 1u; h.g3 -= (uint32_t)G.nx; h.ry = G.hy; }
        return h.g1 >= (uint32_t)G.ny;
    } else {
        const uint32_t nxy = (uint32_t)(G.nx * G.ny);
        if (up) { h.g2 += 1u; h.g3 += nxy; h.rz = 0.0f; } else { h.g2 -= 1u; h.g3 -= nxy; h.rz = G.hz; }
        return h.g2 >= (uint32_t)G.nz;
    }
}

// per-thread counters that live for the whole kernel (flushed once at its end)
struct LaneCounters { unsigned int n_ct = 0, n_dev = 0, n_slab = 0; double incident = 0.0; };

struct NullScorer {
    __device__ __forceinline__ void begin(const Hist &) {}
    __device__ __forceinline__ void deposit(const Hist &, float) {}
    __device__ __forceinline__ void end(const Hist &) {}
};

struct LutShared { const float4 *p; __device__ __forceinline__ float4 operator[](int i) const { return p[i]; } };
struct LutGlobal { const float4 *p; __device__ __forceinline__ float4 operator[](int i) const { return __ldg(p + i); } };

// status of a history after an iteration in the beam line: still inside, on the exit plane of its device, or ended
enum : int { BEAM_CONT = 0, BEAM_EXIT = 1, BEAM_STOPPED = 2, BEAM_NUCLEAR = 3, BEAM_ESCAPED = 4 };

// The beam line is cut into STAGES, each run by its own kernel so that a warp only ever holds histories that execute the
// same code:
//   rs_enter  + rs_iter   range shifter: vacuum drift to its entrance (once), then one slab step per iteration;
//   ap_enter              vacuum drift to the aperture entrance and the OPENING PHASE: the per-step medium test of P:L87
//                         and the drifts through the opening, until a brass step is due or the exit plane is reached --
//                         run converged, one thread per history, by source_kernel / ap_entry_kernel;
//   ap_iter               one iteration inside the aperture region: brass slab step (the opening phase again only for
//                         the few histories that scatter back into the opening).
// beam_step() strings the same functions together for the trace kernels, so a trace records exactly what the production
// kernels compute.

// slab geometry, common to range shifter and aperture region: distance to the exit plane, fixed step (C4: d = min(s_rs |
// s_ap, distance to the exit plane))
struct SlabGeom { float w_in, T, d; bool ex; };

__device__ __forceinline__ void slab_geometry(const DevParams &P, const DevBeam *bp, bool rs, const Hist &h, SlabGeom &g)
{
    const float *wp = rs ? &bp->w_rs_in : &bp->w_ap_in;
    g.w_in = __ldg(wp);
    g.T = __ldg(wp + 1) - g.w_in;
    g.d = rs ? P.s_rs : P.s_ap; g.ex = false;
    const float rem = g.T - h.rz;
    if (rem <= g.d * h.uz) { g.d = fmaxf(__fdiv_rn(rem, h.uz), 0.0f); g.ex = true; }
}

// one slab step (range shifter or brass): C4 items 1-8 and 10.  `out` = the history reached the exit plane of the device.
template <int FL, class Tracer>
__device__ __forceinline__ int slab_step(const Ctx &c, Hist &h, const Medium &m, const SlabGeom &g, int reg, float &dep,
                                         LaneCounters &lc, Tracer &tr, bool &out)
{
    StepOut o;
    const float Eb = h.E; const uint32_t st = h.step;
    const float lat = fmaxf(fabsf(h.ux), fabsf(h.uy));        // direction of travel during the step
    const int cause = step_physics<FL>(c.P, h, m, g.d, c.K, o);
    h.rx = fmaf(-o.s, lat, h.rx);                              // brass budget (meaningless, and unused, in the range shifter)
    if (cause == CONT) {
        // C4-8: move along the OLD direction, then rotate
        pair_axpy(h.g0, h.g1, o.s, h.ux, h.lx);
        pair_axpy(h.g2, h.g3, o.s, h.uy, h.ly);
        h.rz = fmaf(o.s, h.uz, h.rz);
        if (((FL >= 0) ? FL : c.P.flags) & 1) rotate(h, o.theta, o.uphi);
    }
    dep += o.dep;
    lc.n_slab += (cause != STOPPED);
    out = (cause == CONT) && o.on_d && g.ex;
    if (out) h.rz = g.T;
    if (Tracer::on) tr.put(h, beam_xh(h), beam_yh(h), g.w_in + h.rz, st, reg, nullptr, Eb, h.E, o.s, cause, o.dep);
    return cause;
}

// u_w <= 0 inside the beam line ends the history as ESCAPED (C4, last paragraph)
template <class Tracer>
__device__ __forceinline__ int beam_escape(const Hist &h, float w_in, Tracer &tr)
{
    if (Tracer::on) tr.put(h, beam_xh(h), beam_yh(h), w_in + h.rz, h.step, REG_VAC, nullptr, h.E, h.E, 0.0f, ESCAPED);
    return BEAM_ESCAPED;
}

// pending vacuum drift from the start plane to the range-shifter entrance
template <class Tracer>
__device__ __forceinline__ int rs_enter(const Ctx &c, Hist &h, Tracer &tr)
{
    const DevBeam *bp = c.beams + (h.region >> 8);
    const float w1 = __ldg(&bp->w_rs_in), w0 = __ldg(&bp->w_start);
    if (drift_gap(h, w1 - w0, w1, tr) != CONT) return beam_escape(h, w0, tr);
    h.region = REG_RS | (h.region & ~0xff);
    return BEAM_CONT;
}

// one range-shifter step (S2; homogeneous, energy-only medium)
template <int FL, class Tracer>
__device__ __forceinline__ int rs_iter(const Ctx &c, Hist &h, float &dep_rs, LaneCounters &lc, Tracer &tr)
{
    const DevParams &P = c.P;
    const DevBeam *bp = c.beams + (h.region >> 8);
    if (!(h.uz > 0.0f)) return beam_escape(h, __ldg(&bp->w_rs_in), tr);
    SlabGeom g;
    slab_geometry(P, bp, true, h, g);
    const Medium m = { P.rs_rsp, P.rs_inv_rsp, P.rs_rho, P.rs_inv_X0, P.rs_za_rho };
    bool out;
    const int cause = slab_step<FL>(c, h, m, g, REG_RS, dep_rs, lc, tr, out);
    if (__builtin_expect(cause != CONT, 0)) return (cause == NUCLEAR) ? BEAM_NUCLEAR : BEAM_STOPPED;
    if (__builtin_expect(!out, 1)) return BEAM_CONT;
    h.region = (__ldg(&bp->has_ap) ? REG_TO_AP : REG_TO_CT) | (h.region & ~0xff);
    return BEAM_EXIT;
}

// S3, opening phase: the medium under the current (u, v) is tested at the start of every step; in the opening the
// proton drifts with its previous velocity and direction.  Runs until a brass step is due (returns BEAM_CONT; h.rx = lateral
// travel, in mm of the L-infinity norm, over which the history is KNOWN to stay in brass, > 0; g = geometry of that step) or
// the exit plane is reached (BEAM_EXIT, region REG_TO_CT).
// Safe-distance skipping: every tile within Chebyshev distance k - 1 of the current one is fully open, so the next per-step
// tests are known to answer "open" as long as the lateral travel stays below (k - 1) tiles.
template <class Tracer>
__device__ __forceinline__ int ap_open_phase(const Ctx &c, const DevBeam *bp, Hist &h, SlabGeom &g, Tracer &tr)
{
    const DevParams &P = c.P;
    const float T = g.T, w_in = g.w_in;
    for (;;) {
        float safe_u, safe_v;
        if (!aperture_query(bp, beam_xh(h), beam_yh(h), safe_u, safe_v)) {
            h.rx = fmaxf(fminf(safe_u, safe_v), 1e-30f);          // > 0: the step that follows this test IS a brass step
            return BEAM_CONT;
        }
        // nf = full steps left before the exit step; if all of their tests are known, go straight to the exit plane, else
        // take the known ones (at least one step) and test again.
        const float rem = T - h.rz, duz = P.s_ap * h.uz;
        // nf = number of j >= 0 with rem - j duz > duz (the per-step rule `rem <= d u_w` decides the exit step); the
        // rounded quotient can be off by one when rem / duz sits next to an integer, so it is checked against that rule
        int nf = g.ex ? 0 : max((int)ceilf(__fdiv_rn(rem, duz)) - 1, 0);
        if (!g.ex) {
            if (fmaf(-(float)nf, duz, rem) > duz) nf += 1;
            else if (nf > 0 && fmaf(-(float)(nf - 1), duz, rem) <= duz) nf -= 1;
        }
        float n_safe = 0.0f;
        if (nf > 0 && safe_u > 0.0f && safe_v > 0.0f) {
            const float nu = __fdividef(safe_u, fmaxf(fabsf(P.s_ap * h.ux), 1e-12f));
            const float nv = __fdividef(safe_v, fmaxf(fabsf(P.s_ap * h.uy), 1e-12f));
            n_safe = floorf(fminf(fminf(nu, nv), 65536.0f));
        }
        const bool whole = n_safe >= (float)nf;            // includes the plain exit step (nf = 0)
        const int n = whole ? nf : max((int)n_safe, 1);    // full steps taken now
        if (Tracer::on && n > 0) {     // the same arithmetic, one record per full step
            const uint32_t g0 = h.g0, g1 = h.g1, g2 = h.g2, g3 = h.g3; const float rz0 = h.rz;
            for (int j = 1; j <= n; ++j) {
                const float sj = (float)j * P.s_ap;
                h.g0 = g0; h.g1 = g1; h.g2 = g2; h.g3 = g3;
                pair_axpy(h.g0, h.g1, sj, h.ux, h.lx); pair_axpy(h.g2, h.g3, sj, h.uy, h.ly);
                h.rz = fmaf(sj, h.uz, rz0);
                tr.put(h, beam_xh(h), beam_yh(h), w_in + h.rz, h.step + (uint32_t)(j - 1), REG_AP_OPEN, nullptr, h.E, h.E, P.s_ap, CONT);
            }
            h.g0 = g0; h.g1 = g1; h.g2 = g2; h.g3 = g3; h.rz = rz0;
        }
        if (whole) {
            const float rz_nf = fmaf((float)nf * P.s_ap, h.uz, h.rz);                  // depth after the full steps
            const float d_exit = fmaxf(__fdiv_rn(T - rz_nf, h.uz), 0.0f);
            const float s_tot = fmaf((float)nf, P.s_ap, d_exit);
            pair_axpy(h.g0, h.g1, s_tot, h.ux, h.lx); pair_axpy(h.g2, h.g3, s_tot, h.uy, h.ly);
            h.rz = T;
            h.step += (uint32_t)(nf + 1);
            if (Tracer::on) tr.put(h, beam_xh(h), beam_yh(h), w_in + T, h.step - 1u, REG_AP_OPEN, nullptr, h.E, h.E, d_exit, CONT);
            h.region = REG_TO_CT | (h.region & ~0xff);
            return BEAM_EXIT;
        }
        const float sn = (float)n * P.s_ap;
        pair_axpy(h.g0, h.g1, sn, h.ux, h.lx); pair_axpy(h.g2, h.g3, sn, h.uy, h.ly);
        h.rz = fmaf(sn, h.uz, h.rz);
        h.step += (uint32_t)n;
        // geometry of the next step
        g.d = P.s_ap; g.ex = false;
        const float rem2 = T - h.rz;
        if (rem2 <= g.d * h.uz) { g.d = fmaxf(__fdiv_rn(rem2, h.uz), 0.0f); g.ex = true; }
    }
}

// pending vacuum drift to the aperture entrance + the opening phase from there.  BEAM_EXIT: clean transit (region
// REG_TO_CT); BEAM_CONT: the history stands in the aperture region and its next step is a brass step (h.rx > 0).
template <class Tracer>
__device__ __forceinline__ int ap_enter(const Ctx &c, Hist &h, Tracer &tr)
{
    const DevBeam *bp = c.beams + (h.region >> 8);
    const float w1 = __ldg(&bp->w_ap_in);
    const float w0 = __ldg(&bp->has_rs) ? __ldg(&bp->w_rs_out) : __ldg(&bp->w_start);
    if (drift_gap(h, w1 - w0, w1, tr) != CONT) return beam_escape(h, w0, tr);
    h.region = REG_AP | (h.region & ~0xff);
    h.rx = 0.0f;
    SlabGeom g;
    slab_geometry(c.P, bp, false, h, g);
    return ap_open_phase(c, bp, h, g, tr);
}

// One iteration of a history that stands in the aperture region (S3): the opening phase if its medium is not known to be
// brass, then at most ONE brass step.  `conv` = the lanes of the warp that called together: they re-converge before the
// expensive slab step, whatever the opening phase did (0 = no forced re-convergence, for one-thread-per-history callers).
// dep_ap = energy deposited so far in the brass.
template <int FL, class Tracer>
__device__ __forceinline__ int ap_iter(const Ctx &c, Hist &h, float &dep_ap, LaneCounters &lc, Tracer &tr, unsigned conv)
{
    const DevParams &P = c.P;
    const DevBeam *bp = c.beams + (h.region >> 8);
    int status = BEAM_CONT;
    bool do_step = false;
    SlabGeom g = { __ldg(&bp->w_ap_in), 0.0f, 0.0f, false };
    if (!(h.uz > 0.0f)) status = beam_escape(h, g.w_in, tr);
    else {
        slab_geometry(P, bp, false, h, g);
        do_step = h.rx > 0.0f;             // while the budget is positive the per-step test of P:L87 can only answer "brass"
        if (!do_step) { status = ap_open_phase(c, bp, h, g, tr); do_step = status == BEAM_CONT; }
    }
    if (conv) __syncwarp(conv);
    if (do_step) {
        const Medium m = { P.brass_rsp, P.brass_inv_rsp, P.brass_rho, P.brass_inv_X0, P.brass_za_rho };
        bool out;
        const int cause = slab_step<FL>(c, h, m, g, REG_AP, dep_ap, lc, tr, out);
        if (cause != CONT) status = (cause == NUCLEAR) ? BEAM_NUCLEAR : BEAM_STOPPED;
        else if (out) { h.region = REG_TO_CT | (h.region & ~0xff); status = BEAM_EXIT; }
    }
    return status;
}

// One iteration of history h anywhere in the beam line (trace kernels): pending drifts, then the stage's own iteration.
// Returns the BEAM_* status; when the history ended, h.region holds the region it ended in and h.E the energy it had left.
// Nothing is tallied here: the once-per-history bookkeeping is done by book_beam_end().
template <class Tracer>
__device__ __forceinline__ int beam_step(const Ctx &c, Hist &h, float &dep_rs, float &dep_ap, LaneCounters &lc, Tracer &tr)
{
    int reg = h.region & 0xff;
    if (reg == REG_TO_CT) return BEAM_EXIT;              // no device at all
    if (reg == REG_TO_RS) {
        if (rs_enter(c, h, tr) != BEAM_CONT) return BEAM_ESCAPED;
        reg = REG_RS;
    }
    if (reg == REG_RS) {
        const int st = rs_iter<-1>(c, h, dep_rs, lc, tr);
        if (st != BEAM_EXIT) return st;
        return ((h.region & 0xff) == REG_TO_CT) ? BEAM_EXIT : BEAM_CONT;      // the aperture follows
    }
    if (reg == REG_TO_AP) {
        const int st = ap_enter(c, h, tr);
        if (st != BEAM_CONT) return st;
    }
    return ap_iter<-1>(c, h, dep_ap, lc, tr, 0u);
}

// ---- once-per-history bookkeeping (tallies of S:8b), done in the kernels' event passes by ALL 32 lanes of the warp together:
// the lanes with something to book contribute to a shuffle reduction and lane 0 adds the sum to the warp's own slot in
// shared memory (fp64 atomics on shared memory are compare-and-swap loops that serialise the contributing lanes)
__device__ __forceinline__ void warp_book_d(WarpTally *w, int lane, int k, bool on, float v)
{
    if (__ballot_sync(0xffffffffu, on && v != 0.0f) == 0u) return;
    double s = on ? (double)v : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) w->d[k] += s;
}
__device__ __forceinline__ void warp_book_c(WarpTally *w, int lane, int k, bool on)
{
    const unsigned m = __ballot_sync(0xffffffffu, on);
    if (m != 0u && lane == 0) w->c[k] += (unsigned)__popc(m);
}

// beam line: `due` = this lane holds a finished history whose bookkeeping is due (status != BEAM_CONT); dep = the energy it
// deposited in this stage's device (tally k_dep = TD_DEP_RS | TD_DEP_BRASS)
__device__ __forceinline__ void book_beam_end(const DevParams &P, const Hist &h, bool due, int status, float dep, int k_dep,
                                              LaneCounters &lc, WarpTally *w, int lane)
{
    warp_book_d(w, lane, k_dep, due, dep);
    const bool ended = due && status != BEAM_EXIT;       // the beam-line steps of a survivor are booked at the CT entry
    if (ended) lc.n_dev += h.step;
    const bool nuc = ended && status == BEAM_NUCLEAR, stop = ended && status == BEAM_STOPPED, esc = ended && status == BEAM_ESCAPED;
    warp_book_d(w, lane, TD_REMOVED, nuc, (1.0f - P.gamma_loc) * h.E);
    warp_book_c(w, lane, TC_NUCLEAR, nuc);
    warp_book_c(w, lane, k_dep == TD_DEP_RS ? TC_STOP_RS : TC_STOP_BRASS, stop);
    warp_book_d(w, lane, TD_ESCAPED, esc, h.E);
    warp_book_c(w, lane, TC_ESCAPED, esc);
}

// CT entry of a history that left the beam line (region REG_TO_CT): books the beam-line step count and, on a miss,
// the escape.  Returns CONT or ESCAPED.
template <class Sink, class Tracer>
__device__ __forceinline__ int ct_entry(const Ctx &c, Hist &h, LaneCounters &lc, const Sink &sink, Tracer &tr)
{
    const DevBeam *bp = c.beams + (h.region >> 8);
    const float w_now = __ldg(&bp->has_ap) ? __ldg(&bp->w_ap_out) : (__ldg(&bp->has_rs) ? __ldg(&bp->w_rs_out) : __ldg(&bp->w_start));
    const int ec = enter_ct(c, *bp, w_now, h, tr);
    lc.n_dev += h.step;
    h.region = REG_CT | (h.region & ~0xff);
    if (ec != CONT) { sink.add_d(TD_ESCAPED, h.E); sink.add_c(TC_ESCAPED, 1u); }
    return ec;
}

// One voxel step of history h (S4, S5, S6/S7).  Returns CONT or the cause that ended the history; the once-per-history
// tallies are booked by book_ct_end() in the kernel's refill pass.  hdep = energy deposited in the CT so far.
// hu_pre (optional): the HU of the voxel the history stands in, fetched by the caller at the end of the previous step (the
// voxel kernel does: HU -> table is a chain of two dependent loads at the head of the step, 6 % of its stall samples).
template <int FL, class Lut, class Scorer, class Tracer>
__device__ __forceinline__ int ct_step(const Ctx &c, const Lut &lut, Hist &h, float &hdep, LaneCounters &lc,
                                       Scorer &sc, Tracer &tr, const int *hu_pre = nullptr)
{
    const DevParams &P = c.P;
    const DevGrid &G = c.G;
    int ax; bool up;
    const float d = face_distance(G, h, ax, up);
    int t = (hu_pre ? *hu_pre : (int)__ldg(c.hu + h.g3)) - G.hu_min;
    t = min(max(t, 0), G.n_lut - 1);
    const float4 mv = lut[t];                 // rsp, rho, xsp / X0_w, 1 / rsp
    const Medium m = { mv.x * c.rsp_scale, mv.w * c.inv_rsp_scale, mv.y, mv.z, P.za_w * mv.y };
    StepOut o;
    const float Eb = h.E; const uint32_t st = h.step;
    int cause = step_physics<FL>(P, h, m, d, c.K, o);
    if (cause == CONT) {
        // C4-8: move along the OLD direction, then rotate
        h.rx = fmaf(o.s, h.lx, fmaf(o.s, h.ux, h.rx));
        h.ry = fmaf(o.s, h.ly, fmaf(o.s, h.uy, h.ry));
        h.rz = fmaf(o.s, h.lz, fmaf(o.s, h.uz, h.rz));
        if (((FL >= 0) ? FL : P.flags) & 1) rotate(h, o.theta, o.uphi);
    }
    hdep += o.dep;
    if (o.dep != 0.0f) sc.deposit(h, o.dep);      // S6 / S7: the voxel at the START of the step
    const int iv0[3] = { (int)h.g0, (int)h.g1, (int)h.g2 };
    if (cause == CONT && o.on_d && cross_face(G, h, ax, up)) cause = ESCAPED;
    lc.n_ct += (cause != STOPPED);
    if (Tracer::on) tr.put(h, fmaf((float)(int)h.g0, G.hx, G.ox) + h.rx, fmaf((float)(int)h.g1, G.hy, G.oy) + h.ry,
                           fmaf((float)(int)h.g2, G.hz, G.oz) + h.rz, st, REG_CT, iv0, Eb, h.E, o.s, cause, o.dep);
    return cause;
}

// CT stage: `due` = this lane holds a finished history (cause != CONT); hdep = energy it deposited in the CT
__device__ __forceinline__ void book_ct_end(const DevParams &P, const Hist &h, bool due, int cause, float hdep, WarpTally *w, int lane)
{
    warp_book_d(w, lane, TD_DEP_CT, due, hdep);
    const bool nuc = due && cause == NUCLEAR, esc = due && cause == ESCAPED;
    warp_book_d(w, lane, TD_REMOVED, nuc, (1.0f - P.gamma_loc) * h.E);
    warp_book_c(w, lane, TC_NUCLEAR, nuc);
    warp_book_d(w, lane, TD_ESCAPED, esc, h.E);
    warp_book_c(w, lane, TC_ESCAPED, esc);
    warp_book_c(w, lane, TC_STOP_CT, due && !nuc && !esc);
}

}  // namespace vpk
