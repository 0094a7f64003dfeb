/*
 * vpmc_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded CPU oracle of the VPMC transport-and-scoring
 * loop with aperture block (arXiv 2307.01416).  fp64 state arithmetic, one
 * history at a time, in the order and notation of SURVEY.md section 8(c)
 * (C0..C6), which is the written-out closed-form reading of the passages
 *   P:L73  one particle type, all initialised up front, identical logic
 *   P:L75  per-step lookup X(E): deposited energy, straggling, deflection,
 *          interaction probability
 *   P:L81  30 mm brass block, stops ~155 MeV, downstream face 150 mm to
 *          isocentre; range shifter WET 45 mm, downstream face 190 mm
 *   P:L83  range shifter = homogeneous, energy-only medium
 *   P:L87  aperture: per-MC-step opening test; opening -> "transported with
 *          the previous velocity and direction"; brass -> brass physics
 *   P:L160 scenarios: RSP scaling, isocentre shifts
 * (P:Lnn = /root/reference/PAPER.md line nn.)  Every reading of a point on
 * which the paper is silent is listed in DESIGN.md section 3.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this file.  It shares no code, header,
 * table or constant generator with the CUDA path under
 * paper_2307_01416_b200/csrc/.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): Philox known answers; CSDA
 * range = alpha E^p; closed-form depth dose; Highland slab angle; Fermi-Eyges
 * lateral sigma; Bohr range straggling; nuclear survival 1/(1+beta R0);
 * energy bookkeeping; closed brass block; range-shifter exit energies;
 * DDA vs dense micro-stepping; hand-traced histories on a 4^3 grid; shift /
 * RSP-scale scenario identities; CSR brute force.
 * Parity unpinned: absolute agreement with the paper's own VPMC / MCsquare /
 * RayStation doses (none of them is available).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_MP 938.272            /* proton rest energy, MeV (C4-4, C4-7) */
#define ORC_TWO_PI 6.283185307179586476925286766559
#define ORC_MEV_PER_G_TO_GY 1.602176634e-10 /* C6 */

#define ORC_FLAG_MCS 1
#define ORC_FLAG_STRAGGLE 2
#define ORC_FLAG_NUCLEAR 4

enum { ORC_REG_VAC = 0, ORC_REG_RS = 1, ORC_REG_AP_OPEN = 2, ORC_REG_AP_BRASS = 3, ORC_REG_CT = 4 };
enum { ORC_CONT = 0, ORC_STOPPED = 1, ORC_NUCLEAR = 2, ORC_ESCAPED = 3 };

/* C0: parameters */
typedef struct {
    double alpha, p;            /* Bragg-Kleeman R = alpha E^p (mm, MeV) */
    double X0_w;                /* radiation length of water, mm */
    double Es, c_log;           /* Highland constants */
    double beta_nuc, gamma_loc; /* nuclear slope per mm, locally absorbed fraction */
    double k_bohr, za_w;        /* Bohr variance constant, Z/A of water */
    double R_cut, f_R, s_max;   /* stop range, max fraction of R per step, geometric cap */
    double s_rs, s_ap;          /* fixed geometric steps in range shifter / aperture */
    double brass_rsp, brass_rho, brass_X0, brass_za;
    double rs_rsp, rs_rho, rs_X0;
    double rho_min;             /* density floor in the dose conversion */
    double delta_E;             /* relative source energy spread */
    int32_t flags;
    int32_t n_batches;
} orc_params;

typedef struct {
    int32_t n[3];
    double h[3];
    double origin[3];           /* low corner of voxel (0,0,0), CT frame, mm */
    const int16_t *hu;          /* v = ix + nx*(iy + ny*iz) */
} orc_ct;

typedef struct {
    int32_t n;                  /* nodes ascending in hu */
    const double *hu, *rsp, *rho, *xsp; /* xsp may be NULL -> rho */
} orc_calib;

typedef struct {
    double iso[3];
    double rot[9];              /* r_ct = iso + rot * r_beam, row-major */
    int32_t n_spots;
    const double *x, *y, *E, *w, *sigma;
    double rs_wet;              /* 0 = no range shifter */
    double rs_face;             /* downstream face, mm upstream of isocentre (190) */
    int32_t ap_present;
    double ap_T, ap_face;       /* thickness; downstream face mm upstream of isocentre (150) */
    const uint8_t *ap_open;     /* ny*nx, 1 = open */
    int32_t ap_nx, ap_ny;
    double ap_u0, ap_v0, ap_du, ap_dv;
    /* the opening as the paper describes it ("the opening boundary ... polygon", crossing-number test,
     * ref. 67).  ap_n_poly > 0: the opening is the closed polygon of these vertices (x0, y0, x1, y1, ...; beam frame, mm)
     * and the bitmap is not used. */
    int32_t ap_n_poly;
    const double *ap_poly;
} orc_beam;

typedef struct {
    orc_params P;
    orc_ct ct;
    orc_calib cal;
    int32_t n_beams;
    const orc_beam *beams;
} orc_problem;

typedef struct { double shift[3]; double rsp_scale; } orc_scenario;

typedef struct {
    double incident, dep_ct, dep_rs, dep_brass, escaped, removed;
    uint64_t n_stopped_ct, n_stopped_rs, n_stopped_brass, n_nuclear, n_escaped;
} orc_tallies;

typedef struct {
    uint64_t hid;
    int32_t step, region, cause;
    int32_t ivox[3];            /* voxel at step start (CT) else -1 */
    double r[3], u[3];          /* after the step; beam frame in the beam line, CT frame from the CT-entry drift on */
    double E_before, E_after, s;
    double t_rad, tau, tau_star; /* carried scattering depth and nuclear optical depth after the step; threshold */
    double dep;                 /* energy deposited in the step's cell (CT voxel, range-shifter or brass tally), MeV */
} orc_step_rec;

/* ------------------------------------------------------------------ C1 */

/* Philox4x32-10 (Salmon et al. 2011), SURVEY 8c-C1. */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* u = (2*(x>>9)+1) * 2^-24: 23 random bits, strictly in (0,1), exact in fp32 */
double orc_u01(uint32_t x)
{
    return (double)(2u * (x >> 9) + 1u) * (1.0 / 16777216.0);
}

/* Test hook (tests/test_oracle_geometry.py, hand-traced histories with MCS on): when set, the
 * transport block (purpose 0) of step k < n is u[4k..4k+3] instead of the Philox output.  No arithmetic here. */
static const double *g_inject_u = NULL;
static int32_t g_inject_n = 0;
void orc_inject_uniforms(const double *u, int32_t n_steps) { g_inject_u = u; g_inject_n = u ? n_steps : 0; }

static void draw4(uint64_t hid, uint32_t step, uint32_t purpose, uint64_t seed, double u[4])
{
    if (purpose == 0u && g_inject_u && step < (uint32_t)g_inject_n) {
        for (int i = 0; i < 4; ++i) u[i] = g_inject_u[4 * (size_t)step + i];
        return;
    }
    uint32_t ctr[4] = { (uint32_t)hid, (uint32_t)(hid >> 32), step, purpose };
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t o[4];
    orc_philox4x32_10(ctr, key, o);
    for (int i = 0; i < 4; ++i) u[i] = orc_u01(o[i]);
}

/* ------------------------------------------------------------------ C2 */

/* Largest-remainder apportionment of N histories to spot weights (C2). */
void orc_apportion(uint64_t N, const double *w, int32_t n, uint64_t *counts)
{
    double W = 0.0;
    for (int32_t j = 0; j < n; ++j) W += w[j];
    double *frac = (double *)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
    uint64_t assigned = 0;
    for (int32_t j = 0; j < n; ++j) {
        double q = (W > 0.0) ? (double)N * w[j] / W : 0.0;
        double f = floor(q);
        counts[j] = (uint64_t)f;
        frac[j] = q - f;
        assigned += counts[j];
    }
    uint64_t left = (N > assigned) ? N - assigned : 0;
    while (left > 0) {              /* one each to the largest fractional parts, ties to lower index */
        int32_t best = -1;
        for (int32_t j = 0; j < n; ++j)
            if (frac[j] >= 0.0 && (best < 0 || frac[j] > frac[best])) best = j;
        if (best < 0) {             /* more leftovers than spots: start another round */
            for (int32_t j = 0; j < n; ++j) frac[j] = 0.0;
            if (n == 0) break;
            continue;
        }
        counts[best] += 1;
        frac[best] = -1.0;
        --left;
    }
    free(frac);
}

/* ------------------------------------------------------------------ C5 */

static double pl_interp(const orc_calib *c, const double *y, double hu)
{
    if (hu <= c->hu[0]) return y[0];
    if (hu >= c->hu[c->n - 1]) return y[c->n - 1];
    int32_t k = 0;
    while (k + 2 < c->n && hu >= c->hu[k + 1]) ++k;
    double t = (hu - c->hu[k]) / (c->hu[k + 1] - c->hu[k]);
    return y[k] + t * (y[k + 1] - y[k]);
}

/* HU -> (rsp, rho, xsp), piecewise linear, clamped at the end nodes. */
void orc_calib_eval(const orc_calib *c, double hu, double out[3])
{
    out[0] = pl_interp(c, c->rsp, hu);
    out[1] = pl_interp(c, c->rho, hu);
    out[2] = c->xsp ? pl_interp(c, c->xsp, hu) : out[1];
}

/* ------------------------------------------------------------------ C4 */

typedef struct { double rsp, rho_rel, inv_X0, za_rho; } medium;

typedef struct {
    double r[3], u[3];
    double E, t_rad, tau, tau_star;
    uint32_t step;
} hist;

/* per-history digest (orc_digests): number of records, FNV-1a hash of the discrete trace, state after the last record */
typedef struct {
    uint64_t hid, hash;
    int32_t n_rec, cause;
    double r[3];
    double E_last, dep_ct;
} orc_digest;

typedef struct {
    orc_step_rec *recs; int32_t max, n;
    orc_digest *dig;            /* when set, records are digested instead of stored */
} tracer;

static void fnv_mix(uint64_t *h, uint32_t v) { *h = (*h ^ (uint64_t)v) * 1099511628211ull; }

static void trace_put(tracer *t, uint64_t hid, const hist *h, uint32_t step, int region,
                      const int32_t iv[3], double Eb, double Ea, double s, int cause, double dep)
{
    if (t && t->dig) {          /* hash over (region, cause, ivox[0..2]) of every record, one FNV-1a round per 32-bit word */
        orc_digest *d = t->dig;
        fnv_mix(&d->hash, (uint32_t)region); fnv_mix(&d->hash, (uint32_t)cause);
        for (int a = 0; a < 3; ++a) fnv_mix(&d->hash, (uint32_t)(iv ? iv[a] : -1));
        d->n_rec += 1; d->cause = cause; d->E_last = Ea;
        for (int a = 0; a < 3; ++a) d->r[a] = h->r[a];
        return;
    }
    if (!t || t->n >= t->max) { if (t) t->n++; return; }
    orc_step_rec *q = &t->recs[t->n++];
    q->hid = hid; q->step = (int32_t)step; q->region = region; q->cause = cause;
    for (int a = 0; a < 3; ++a) { q->ivox[a] = iv ? iv[a] : -1; q->r[a] = h->r[a]; q->u[a] = h->u[a]; }
    q->E_before = Eb; q->E_after = Ea; q->s = s;
    q->t_rad = h->t_rad; q->tau = h->tau; q->tau_star = h->tau_star;
    q->dep = dep;
}

static double highland_A(double t, double c_log)
{
    if (t <= 0.0) return 0.0;
    double f = 1.0 + c_log * log(t);
    return t * f * f;
}

/* One material step (C4 items 1-8, 10).  d = geometric limit.  On return
 * *s is the step taken, *dep the energy deposited in the current cell,
 * *removed the energy taken away by a nuclear event, *on_d says the step
 * ended on the geometric limit.  Returns the cause. */
static int material_step(const orc_params *P, hist *h, const medium *m, double d,
                         uint64_t hid, uint64_t seed,
                         double *s_out, double *dep, double *removed, int *on_d)
{
    *removed = 0.0; *on_d = 0;
    const double E = h->E;
    /* 1 */
    const double R = P->alpha * pow(E, P->p);
    if (R <= P->R_cut) { *dep = E; *s_out = 0.0; h->E = 0.0; return ORC_STOPPED; }
    /* 2 */
    double s = d; int face = 1;
    double lim = fmax(P->f_R * R, P->R_cut) / m->rsp;
    if (lim < s) { s = lim; face = 0; }
    if (P->s_max < s) { s = P->s_max; face = 0; }
    const double Rp = R - s * m->rsp;
    const double Ebar = pow(Rp / P->alpha, 1.0 / P->p);
    /* 3 */
    double u[4];
    draw4(hid, h->step, 0u, seed, u);
    /* 4 */
    double Ep = Ebar;
    if (P->flags & ORC_FLAG_STRAGGLE) {
        double Emid = 0.5 * (E + Ebar);
        double g = 1.0 + Emid / ORC_MP;
        double b2 = 1.0 - 1.0 / (g * g);
        double var = P->k_bohr * m->za_rho * s * g * g * (1.0 - 0.5 * b2);
        double z0 = sqrt(-2.0 * log(u[2])) * cos(ORC_TWO_PI * u[3]);
        Ep = Ebar - sqrt(var) * z0;
        if (Ep < 0.0) Ep = 0.0;
        if (Ep > E) Ep = E;
    }
    /* 5 */
    *dep = E - Ep;
    *s_out = s;
    /* 6 */
    if (P->flags & ORC_FLAG_NUCLEAR) {
        h->tau += P->beta_nuc / (1.0 + P->beta_nuc * R) * m->rho_rel * s;
        if (h->tau >= h->tau_star) {
            *dep += P->gamma_loc * Ep;
            *removed = (1.0 - P->gamma_loc) * Ep;
            h->E = Ep;
            return ORC_NUCLEAR;
        }
    }
    /* 7 */
    double theta = 0.0, phi = 0.0;
    if (P->flags & ORC_FLAG_MCS) {
        double tp = h->t_rad + s * m->inv_X0;
        double dA = highland_A(tp, P->c_log) - highland_A(h->t_rad, P->c_log);
        if (dA < 0.0) dA = 0.0;
        double Em = 0.5 * (E + Ep);
        double pv = (Em * Em + 2.0 * Em * ORC_MP) / (Em + ORC_MP);
        double theta0 = P->Es / pv * sqrt(dA);
        theta = theta0 * sqrt(-2.0 * log(u[0]));
        phi = ORC_TWO_PI * u[1];
        h->t_rad = tp;
    }
    /* 8: move along the old direction, then rotate */
    for (int a = 0; a < 3; ++a) h->r[a] += s * h->u[a];
    if (P->flags & ORC_FLAG_MCS) {
        double st = sin(theta), ct = cos(theta), sp = sin(phi), cp = cos(phi);
        double ux = h->u[0], uy = h->u[1], uw = h->u[2];
        double rho2 = ux * ux + uy * uy;   /* = 1 - uw^2 for a unit vector */
        double nx, ny, nw;
        if (rho2 < 1e-10) {
            nx = st * cp; ny = st * sp; nw = (uw < 0.0 ? -ct : ct);
        } else {
            double sq = sqrt(rho2);
            nx = ux * ct + st * (ux * uw * cp - uy * sp) / sq;
            ny = uy * ct + st * (uy * uw * cp + ux * sp) / sq;
            nw = uw * ct - sq * st * cp;
        }
        double nrm = sqrt(nx * nx + ny * ny + nw * nw);
        h->u[0] = nx / nrm; h->u[1] = ny / nrm; h->u[2] = nw / nrm;
    }
    /* 10 */
    h->E = Ep;
    h->step += 1;
    *on_d = face;
    return ORC_CONT;
}

/* ------------------------------------------------------------------ C3 */

typedef struct {
    const orc_problem *pb;
    const orc_scenario *sc;
    uint64_t seed;
    double *edep;               /* dense nvox accumulator (MeV) */
    int64_t *touched; int64_t n_touched, max_touched; /* optional list of first-touched voxels */
    orc_tallies *tal;
    tracer *tr;
} ctx;

static void finish(ctx *c, int cause, int region, double E_left)
{
    orc_tallies *t = c->tal;
    if (!t) return;
    if (cause == ORC_ESCAPED) { t->escaped += E_left; t->n_escaped++; }
    else if (cause == ORC_NUCLEAR) { t->n_nuclear++; }
    else if (cause == ORC_STOPPED) {
        if (region == ORC_REG_CT) t->n_stopped_ct++;
        else if (region == ORC_REG_RS) t->n_stopped_rs++;
        else t->n_stopped_brass++;
    }
}

/* most upstream w of the (shifted) CT box corners in the beam frame */
static double ct_min_w(const orc_problem *pb, const orc_beam *b, const orc_scenario *sc)
{
    double wmin = INFINITY;
    for (int k = 0; k < 8; ++k) {
        double c[3];
        for (int a = 0; a < 3; ++a) {
            double lo = pb->ct.origin[a], hi = lo + pb->ct.n[a] * pb->ct.h[a];
            c[a] = ((k >> a) & 1 ? hi : lo) - (b->iso[a] - sc->shift[a]);
        }
        /* r_beam = rot^T (r_ct - iso'), w = third component */
        double w = b->rot[2] * c[0] + b->rot[5] * c[1] + b->rot[8] * c[2];
        if (w < wmin) wmin = w;
    }
    return wmin;
}

/* vacuum drift in the beam frame to the plane w = wt (one step, no RNG) */
static int drift_to_plane(ctx *c, hist *h, uint64_t hid, double wt)
{
    if (!(h->u[2] > 0.0)) return ORC_ESCAPED;
    double s = (wt - h->r[2]) / h->u[2];
    if (s < 0.0) s = 0.0;
    h->r[0] += s * h->u[0]; h->r[1] += s * h->u[1]; h->r[2] = wt;
    trace_put(c->tr, hid, h, h->step, ORC_REG_VAC, NULL, h->E, h->E, s, ORC_CONT, 0.0);
    h->step += 1;
    return ORC_CONT;
}

/* P:L87, ref. 67: crossing-number test -- a horizontal ray from (x, y) towards +x crosses the polygon's edges an odd number
 * of times iff the point is inside.  Edge k joins vertex k to vertex k+1 (the last to the first); an edge counts when its
 * end points lie on different sides of the ray's line (y1 > y differs from y2 > y) and it meets that line right of x. */
static int point_in_polygon(const double *xy, int32_t n, double x, double y)
{
    int inside = 0;
    for (int32_t k = 0; k < n; ++k) {
        const double x1 = xy[2 * k], y1 = xy[2 * k + 1];
        const double x2 = xy[2 * ((k + 1) % n)], y2 = xy[2 * ((k + 1) % n) + 1];
        if ((y1 > y) != (y2 > y)) {
            const double xi = x1 + (y - y1) * (x2 - x1) / (y2 - y1);
            if (x < xi) inside = !inside;
        }
    }
    return inside;
}
int orc_point_in_polygon(const double *xy, int32_t n, double x, double y) { return point_in_polygon(xy, n, x, y); }

static void run_history(ctx *c, uint64_t hid, const orc_beam *b, int32_t j)
{
    const orc_problem *pb = c->pb;
    const orc_params *P = &pb->P;
    const orc_scenario *sc = c->sc;
    hist h;
    double u4[4];

    /* C2: source */
    draw4(hid, 0u, 1u, c->seed, u4);
    {
        double rho = sqrt(-2.0 * log(u4[0]));
        double z0 = rho * cos(ORC_TWO_PI * u4[1]), z1 = rho * sin(ORC_TWO_PI * u4[1]);
        double zE = sqrt(-2.0 * log(u4[2])) * cos(ORC_TWO_PI * u4[3]);
        h.r[0] = b->x[j] + b->sigma[j] * z0;
        h.r[1] = b->y[j] + b->sigma[j] * z1;
        h.E = b->E[j] * (1.0 + P->delta_E * zE);
    }
    draw4(hid, 0u, 2u, c->seed, u4);
    h.tau_star = -log(u4[0]);
    h.tau = 0.0; h.t_rad = 0.0; h.step = 0u;
    h.u[0] = 0.0; h.u[1] = 0.0; h.u[2] = 1.0;
    if (c->tal) c->tal->incident += h.E;

    /* C3: regions along w */
    const int has_rs = b->rs_wet > 0.0, has_ap = b->ap_present != 0;
    const double w_rs_out = -b->rs_face, w_rs_in = w_rs_out - b->rs_wet / P->rs_rsp;
    const double w_ap_out = -b->ap_face, w_ap_in = w_ap_out - b->ap_T;
    double w_start;
    if (has_rs) w_start = w_rs_in - 1.0;
    else if (has_ap) w_start = w_ap_in - 1.0;
    else w_start = ct_min_w(pb, b, sc) - 1.0;
    h.r[2] = w_start;

    double s, dep, rem; int on_d, cause;

    if (has_rs) {
        if (drift_to_plane(c, &h, hid, w_rs_in) != ORC_CONT) goto escaped_beamline;
        medium m = { P->rs_rsp, P->rs_rho, 1.0 / P->rs_X0, P->za_w * P->rs_rho };
        for (;;) {
            if (!(h.u[2] > 0.0)) goto escaped_beamline;
            double d = P->s_rs, dist = (w_rs_out - h.r[2]) / h.u[2]; int ex = 0;
            if (dist <= d) { d = dist; ex = 1; }
            if (d < 0.0) d = 0.0;
            double Eb = h.E; uint32_t st = h.step;
            cause = material_step(P, &h, &m, d, hid, c->seed, &s, &dep, &rem, &on_d);
            if (c->tal) { c->tal->dep_rs += dep; c->tal->removed += rem; }
            if (cause == ORC_CONT && on_d && ex) h.r[2] = w_rs_out;
            trace_put(c->tr, hid, &h, st, ORC_REG_RS, NULL, Eb, h.E, s, cause, dep);
            if (cause != ORC_CONT) { finish(c, cause, ORC_REG_RS, 0.0); return; }
            if (on_d && ex) break;
        }
    }
    if (has_ap) {
        if (drift_to_plane(c, &h, hid, w_ap_in) != ORC_CONT) goto escaped_beamline;
        medium m = { P->brass_rsp, P->brass_rho, 1.0 / P->brass_X0, P->brass_za * P->brass_rho };
        for (;;) {
            if (!(h.u[2] > 0.0)) goto escaped_beamline;
            double d = P->s_ap, dist = (w_ap_out - h.r[2]) / h.u[2]; int ex = 0;
            if (dist <= d) { d = dist; ex = 1; }
            if (d < 0.0) d = 0.0;
            /* per-step test of the medium under the current (u,v) */
            int open = 0;
            if (b->ap_n_poly > 0) open = point_in_polygon(b->ap_poly, b->ap_n_poly, h.r[0], h.r[1]);
            else {
                double fx = floor((h.r[0] - b->ap_u0) / b->ap_du), fy = floor((h.r[1] - b->ap_v0) / b->ap_dv);
                if (fx >= 0.0 && fx < (double)b->ap_nx && fy >= 0.0 && fy < (double)b->ap_ny)
                    open = b->ap_open[(int64_t)fy * b->ap_nx + (int64_t)fx] != 0;
            }
            if (open) {   /* "transported with the previous velocity and direction" */
                for (int a = 0; a < 3; ++a) h.r[a] += d * h.u[a];
                if (ex) h.r[2] = w_ap_out;
                trace_put(c->tr, hid, &h, h.step, ORC_REG_AP_OPEN, NULL, h.E, h.E, d, ORC_CONT, 0.0);
                h.step += 1;
                if (ex) break;
                continue;
            }
            double Eb = h.E; uint32_t st = h.step;
            cause = material_step(P, &h, &m, d, hid, c->seed, &s, &dep, &rem, &on_d);
            if (c->tal) { c->tal->dep_brass += dep; c->tal->removed += rem; }
            if (cause == ORC_CONT && on_d && ex) h.r[2] = w_ap_out;
            trace_put(c->tr, hid, &h, st, ORC_REG_AP_BRASS, NULL, Eb, h.E, s, cause, dep);
            if (cause != ORC_CONT) { finish(c, cause, ORC_REG_AP_BRASS, 0.0); return; }
            if (on_d && ex) break;
        }
    }

    /* beam frame -> CT frame (setup shift moves the patient, devices ride on the nozzle) */
    {
        double rb[3] = { h.r[0], h.r[1], h.r[2] }, ub[3] = { h.u[0], h.u[1], h.u[2] };
        for (int a = 0; a < 3; ++a) {
            h.r[a] = (b->iso[a] - sc->shift[a]) + b->rot[3 * a] * rb[0] + b->rot[3 * a + 1] * rb[1] + b->rot[3 * a + 2] * rb[2];
            h.u[a] = b->rot[3 * a] * ub[0] + b->rot[3 * a + 1] * ub[1] + b->rot[3 * a + 2] * ub[2];
        }
    }
    const orc_ct *ct = &pb->ct;
    int32_t iv[3];
    {   /* ray-box entry, slab method; ties to the lowest axis */
        double t_in = 0.0, t_out = INFINITY; int ax = -1, miss = 0;
        for (int a = 0; a < 3; ++a) {
            double lo = ct->origin[a], hi = lo + ct->n[a] * ct->h[a];
            if (h.u[a] == 0.0) { if (h.r[a] < lo || h.r[a] >= hi) miss = 1; continue; }
            double t1 = (lo - h.r[a]) / h.u[a], t2 = (hi - h.r[a]) / h.u[a];
            double tn = t1 < t2 ? t1 : t2, tf = t1 < t2 ? t2 : t1;
            if (tn > t_in) { t_in = tn; ax = a; }
            if (tf < t_out) t_out = tf;
        }
        if (miss || !(t_in < t_out)) {
            trace_put(c->tr, hid, &h, h.step, ORC_REG_VAC, NULL, h.E, h.E, 0.0, ORC_ESCAPED, 0.0);
            finish(c, ORC_ESCAPED, ORC_REG_VAC, h.E); return;
        }
        for (int a = 0; a < 3; ++a) h.r[a] += t_in * h.u[a];
        for (int a = 0; a < 3; ++a) {
            double lo = ct->origin[a], hi = lo + ct->n[a] * ct->h[a];
            if (a == ax) {
                if (h.u[a] > 0.0) { iv[a] = 0; h.r[a] = lo; } else { iv[a] = ct->n[a] - 1; h.r[a] = hi; }
            } else {
                double f = floor((h.r[a] - lo) / ct->h[a]);
                if (f < 0.0) f = 0.0;
                if (f > (double)(ct->n[a] - 1)) f = (double)(ct->n[a] - 1);
                iv[a] = (int32_t)f;
            }
        }
        trace_put(c->tr, hid, &h, h.step, ORC_REG_VAC, NULL, h.E, h.E, t_in, ORC_CONT, 0.0);
        h.step += 1;
    }

    for (;;) {
        /* S4: distance to the nearest voxel face, ties to the lowest axis */
        double d = INFINITY; int ax = -1;
        for (int a = 0; a < 3; ++a) {
            double da;
            if (h.u[a] > 0.0) da = (ct->origin[a] + (double)(iv[a] + 1) * ct->h[a] - h.r[a]) / h.u[a];
            else if (h.u[a] < 0.0) da = (ct->origin[a] + (double)iv[a] * ct->h[a] - h.r[a]) / h.u[a];
            else continue;
            if (da < d) { d = da; ax = a; }
        }
        if (d < 0.0) d = 0.0;
        int64_t v = iv[0] + (int64_t)ct->n[0] * (iv[1] + (int64_t)ct->n[1] * iv[2]);
        double cal[3];
        orc_calib_eval(&pb->cal, (double)ct->hu[v], cal);
        medium m = { cal[0] * sc->rsp_scale, cal[1], cal[2] / P->X0_w, P->za_w * cal[1] };
        double Eb = h.E; uint32_t st = h.step; int32_t iv0[3] = { iv[0], iv[1], iv[2] };
        const int up = ax >= 0 && h.u[ax] > 0.0;   /* direction of travel during the step (C4-8: old direction) */
        cause = material_step(P, &h, &m, d, hid, c->seed, &s, &dep, &rem, &on_d);
        if (c->edep) {
            if (c->touched && c->edep[v] == 0.0 && dep != 0.0 && c->n_touched < c->max_touched) c->touched[c->n_touched++] = v;
            c->edep[v] += dep;
        }
        if (c->tal) { c->tal->dep_ct += dep; c->tal->removed += rem; }
        int out = 0;
        if (cause == ORC_CONT && on_d) {   /* C4-9 */
            if (up) { h.r[ax] = ct->origin[ax] + (double)(iv[ax] + 1) * ct->h[ax]; iv[ax] += 1; }
            else { h.r[ax] = ct->origin[ax] + (double)iv[ax] * ct->h[ax]; iv[ax] -= 1; }
            if (iv[ax] < 0 || iv[ax] >= ct->n[ax]) out = 1;
        }
        if (out) cause = ORC_ESCAPED;
        trace_put(c->tr, hid, &h, st, ORC_REG_CT, iv0, Eb, h.E, s, cause, dep);
        if (cause != ORC_CONT) { finish(c, cause, ORC_REG_CT, cause == ORC_ESCAPED ? h.E : 0.0); return; }
    }

escaped_beamline:
    trace_put(c->tr, hid, &h, h.step, ORC_REG_VAC, NULL, h.E, h.E, 0.0, ORC_ESCAPED, 0.0);
    finish(c, ORC_ESCAPED, ORC_REG_VAC, h.E);
}

/* ------------------------------------------------ history id -> spot (C2) */

typedef struct { int32_t n; uint64_t *start; int32_t *beam; int32_t *local; } spotmap;

static int32_t total_spots(const orc_problem *pb)
{
    int32_t n = 0;
    for (int32_t b = 0; b < pb->n_beams; ++b) n += pb->beams[b].n_spots;
    return n;
}

/* dose mode: start[j] = first history id of global spot j; start[n] = N */
static spotmap build_spotmap(const orc_problem *pb, uint64_t N)
{
    spotmap m; m.n = total_spots(pb);
    m.start = (uint64_t *)calloc((size_t)m.n + 1, sizeof(uint64_t));
    m.beam = (int32_t *)calloc((size_t)m.n + 1, sizeof(int32_t));
    m.local = (int32_t *)calloc((size_t)m.n + 1, sizeof(int32_t));
    double *w = (double *)calloc((size_t)m.n + 1, sizeof(double));
    uint64_t *cnt = (uint64_t *)calloc((size_t)m.n + 1, sizeof(uint64_t));
    int32_t g = 0;
    for (int32_t b = 0; b < pb->n_beams; ++b)
        for (int32_t j = 0; j < pb->beams[b].n_spots; ++j, ++g) { w[g] = pb->beams[b].w[j]; m.beam[g] = b; m.local[g] = j; }
    orc_apportion(N, w, m.n, cnt);
    for (g = 0; g < m.n; ++g) m.start[g + 1] = m.start[g] + cnt[g];
    free(w); free(cnt);
    return m;
}
static void free_spotmap(spotmap *m) { free(m->start); free(m->beam); free(m->local); }

/* counts per global spot for N histories (exported for the tests) */
void orc_spot_counts(const orc_problem *pb, uint64_t N, uint64_t *counts)
{
    spotmap m = build_spotmap(pb, N);
    for (int32_t g = 0; g < m.n; ++g) counts[g] = m.start[g + 1] - m.start[g];
    free_spotmap(&m);
}

static void run_spot_range(ctx *c, const spotmap *m, int32_t g, uint64_t a, uint64_t b, uint64_t hid_offset)
{
    const orc_beam *bm = &c->pb->beams[m->beam[g]];
    for (uint64_t hid = a; hid < b; ++hid) run_history(c, hid_offset + hid, bm, m->local[g]);
}

/* Dose mode: transport history ids [hid_begin, hid_end) of an N-history run
 * that belong to batch `batch` of `n_batches` (C6; each spot's contiguous id
 * range is cut into n_batches contiguous sub-ranges, batch b = union over
 * spots of sub-range b -- DESIGN.md reading R7).  n_batches = 1 -> all.
 * hid_offset is added to every id before it keys the random stream (C1): the
 * sequential stopping rule of SURVEY 8(d) runs its k-th 10^6-history batch as
 * ids k 2^32 + i (R15); 0 everywhere else.
 * edep (nvox doubles, MeV) is accumulated into, not zeroed. */
int orc_dose_edep_offset(const orc_problem *pb, const orc_scenario *sc, uint64_t N, uint64_t seed,
                         uint64_t hid_begin, uint64_t hid_end, int32_t batch, int32_t n_batches,
                         uint64_t hid_offset, double *edep, orc_tallies *tal)
{
    if (n_batches < 1 || batch < 0 || batch >= n_batches) return -1;
    spotmap m = build_spotmap(pb, N);
    ctx c = { pb, sc, seed, edep, NULL, 0, 0, tal, NULL };
    for (int32_t g = 0; g < m.n; ++g) {
        uint64_t n = m.start[g + 1] - m.start[g];
        uint64_t lo = m.start[g] + (uint64_t)(((unsigned __int128)n * (uint64_t)batch) / (uint64_t)n_batches);
        uint64_t hi = m.start[g] + (uint64_t)(((unsigned __int128)n * (uint64_t)(batch + 1)) / (uint64_t)n_batches);
        if (lo < hid_begin) lo = hid_begin;
        if (hi > hid_end) hi = hid_end;
        if (lo < hi) run_spot_range(&c, &m, g, lo, hi, hid_offset);
    }
    free_spotmap(&m);
    return 0;
}

int orc_dose_edep(const orc_problem *pb, const orc_scenario *sc, uint64_t N, uint64_t seed,
                  uint64_t hid_begin, uint64_t hid_end, int32_t batch, int32_t n_batches,
                  double *edep, orc_tallies *tal)
{
    return orc_dose_edep_offset(pb, sc, N, seed, hid_begin, hid_end, batch, n_batches, 0, edep, tal);
}

/* C6: dose[v] = scale * E_dep[v] / (max(rho_v, rho_min) * V_vox[cm^3]) * 1.602176634e-10 Gy */
void orc_dose_from_edep(const orc_problem *pb, const double *edep, double scale, double *dose)
{
    const orc_ct *ct = &pb->ct;
    int64_t nv = (int64_t)ct->n[0] * ct->n[1] * ct->n[2];
    double V = ct->h[0] * ct->h[1] * ct->h[2] * 1e-3;
    for (int64_t v = 0; v < nv; ++v) {
        double cal[3];
        orc_calib_eval(&pb->cal, (double)ct->hu[v], cal);
        double rho = cal[1] > pb->P.rho_min ? cal[1] : pb->P.rho_min;
        dose[v] = scale * edep[v] / (rho * V) * ORC_MEV_PER_G_TO_GY;
    }
}

/* Influence mode: column of global spot g: hid = g*hist_per_spot + i (C2).
 * i in [i_begin, i_end).  edep accumulated into. */
int orc_influence_edep(const orc_problem *pb, const orc_scenario *sc, int32_t g, uint32_t hist_per_spot,
                       uint64_t seed, uint32_t i_begin, uint32_t i_end, double *edep, orc_tallies *tal)
{
    int32_t n = total_spots(pb);
    if (g < 0 || g >= n) return -1;
    int32_t b = 0, j = g;
    while (j >= pb->beams[b].n_spots) { j -= pb->beams[b].n_spots; ++b; }
    ctx c = { pb, sc, seed, edep, NULL, 0, 0, tal, NULL };
    for (uint32_t i = i_begin; i < i_end && i < hist_per_spot; ++i)
        run_history(&c, (uint64_t)g * hist_per_spot + i, &pb->beams[b], j);
    return 0;
}

/* Step records of selected histories.  mode 0: dose mode with N = n_or_hps;
 * mode 1: influence mode with hist_per_spot = n_or_hps.  recs holds
 * n*max_steps records; nrec[i] = records history i produced (may exceed
 * max_steps, in which case only the first max_steps were stored). */
int orc_trace(const orc_problem *pb, const orc_scenario *sc, int32_t mode, uint64_t n_or_hps, uint64_t seed,
              const uint64_t *hids, int32_t n, int32_t max_steps, orc_step_rec *recs, int32_t *nrec)
{
    spotmap m; m.n = 0; m.start = NULL; m.beam = NULL; m.local = NULL;
    if (mode == 0) m = build_spotmap(pb, n_or_hps);
    int32_t nsp = total_spots(pb);
    for (int32_t i = 0; i < n; ++i) {
        tracer tr = { recs + (int64_t)i * max_steps, max_steps, 0, NULL };
        ctx c = { pb, sc, seed, NULL, NULL, 0, 0, NULL, &tr };
        int32_t g;
        if (mode == 0) {
            if (hids[i] >= n_or_hps) { nrec[i] = 0; continue; }
            int32_t lo = 0, hi = m.n;       /* largest g with start[g] <= hid */
            while (hi - lo > 1) { int32_t mid = (lo + hi) / 2; if (m.start[mid] <= hids[i]) lo = mid; else hi = mid; }
            g = lo;
            while (g + 1 < m.n && m.start[g + 1] <= hids[i]) ++g;   /* skip empty spots */
        } else {
            g = (int32_t)(hids[i] / n_or_hps);
        }
        if (g < 0 || g >= nsp) { nrec[i] = 0; continue; }
        int32_t b = 0, j = g;
        while (j >= pb->beams[b].n_spots) { j -= pb->beams[b].n_spots; ++b; }
        run_history(&c, hids[i], &pb->beams[b], j);
        nrec[i] = tr.n;
    }
    if (mode == 0) free_spotmap(&m);
    return 0;
}

/* Digests of the contiguous history ids [hid_begin, hid_begin + n) of the N-history dose run (test support: finds
 * the histories whose discrete trace or end point differs between two implementations without storing every step). */
int orc_digests(const orc_problem *pb, const orc_scenario *sc, uint64_t N, uint64_t seed, uint64_t hid_begin, int32_t n,
                orc_digest *out)
{
    spotmap m = build_spotmap(pb, N);
    int32_t g = 0;
    for (int32_t i = 0; i < n; ++i) {
        uint64_t hid = hid_begin + (uint64_t)i;
        if (hid >= N) { free_spotmap(&m); return -1; }
        while (g + 1 < m.n && m.start[g + 1] <= hid) ++g;
        orc_digest *d = &out[i];
        memset(d, 0, sizeof(*d));
        d->hid = hid; d->hash = 1469598103934665603ull;
        tracer tr = { NULL, 0, 0, d };
        orc_tallies tal;
        memset(&tal, 0, sizeof(tal));
        ctx c = { pb, sc, seed, NULL, NULL, 0, 0, &tal, &tr };
        run_history(&c, hid, &pb->beams[m.beam[g]], m.local[g]);
        d->dep_ct = tal.dep_ct;
    }
    free_spotmap(&m);
    return 0;
}

/* C6 / S8: one CSR row from a dense fp32 column: keep val >= rel_thr*max and
 * val > 0, voxel index ascending.  idx/val may be NULL to count only.
 * The threshold product is taken in fp32 (same precision as the kernel). */
int64_t orc_csr_row(const float *col, int64_t nvox, float rel_thr, int32_t *idx, float *val)
{
    float mx = 0.0f;
    for (int64_t v = 0; v < nvox; ++v) if (col[v] > mx) mx = col[v];
    volatile float thr = rel_thr * mx;
    int64_t k = 0;
    for (int64_t v = 0; v < nvox; ++v) {
        if (col[v] > 0.0f && col[v] >= thr) {
            if (idx) idx[k] = (int32_t)v;
            if (val) val[k] = col[v];
            ++k;
        }
    }
    return k;
}

/* struct sizes, so the ctypes mirror can be checked */
void orc_sizes(int32_t out[8])
{
    out[0] = (int32_t)sizeof(orc_params); out[1] = (int32_t)sizeof(orc_ct); out[2] = (int32_t)sizeof(orc_calib);
    out[3] = (int32_t)sizeof(orc_beam); out[4] = (int32_t)sizeof(orc_problem); out[5] = (int32_t)sizeof(orc_scenario);
    out[6] = (int32_t)sizeof(orc_tallies); out[7] = (int32_t)sizeof(orc_step_rec);
}
