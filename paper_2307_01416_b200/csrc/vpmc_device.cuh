// vpmc_device.cuh -- device-side transport primitives shared by the persistent transport kernel and the trace
// kernel.  Written for sm_100a.  Independent of oracle/ (no shared code or tables).
//
// Physics: SURVEY.md 8(c) C1-C5 (closed-form reading of P:L73-P:L87).  Precision plan:
//   * residual range R in fp64, updated by differences; E re-derived from it every step (MUFU pow);
//   * direction carried as an unevaluated fp32 sum hi + lo (the per-step rotation adds a small increment, so the
//     rounding of the direction no longer random-walks at 6e-8 per step);
//   * beam-frame lateral position as an unevaluated fp32 sum hi + lo as well (the 150-200 mm drifts are long lever
//     arms; fp32 pairs instead of fp64 keep the conversions off the XU pipe), CT position as fp32 LOCAL offsets inside
//     the current voxel; the CT entry itself in fp64, once per history;
//   * Highland's A(t') - A(t) in its difference form (no cancellation);
//   * the random deviates use MUFU intrinsics: they enter as perturbations, never into carried state directly.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace vpk {

constexpr float kMp = 938.272f;
constexpr float kTwoPi = 6.283185307179586f;

// regions of a history.  0-4 are the step-record codes of include/vpmc.h; 5-7 are pending transitions.
enum : int { REG_VAC = 0, REG_RS = 1, REG_AP_OPEN = 2, REG_AP = 3, REG_CT = 4, REG_TO_RS = 5, REG_TO_AP = 6, REG_TO_CT = 7 };
constexpr int REG_AP_BRASS = 3;
enum : int { CONT = 0, STOPPED = 1, NUCLEAR = 2, ESCAPED = 3 };

// Parameters in device form (kernel argument -> constant bank).
struct DevParams {
    float alpha, p, inv_p, inv_alpha;
    float inv_X0_w, Es, c_log;
    float beta_nuc, gamma_loc, k_bohr, za_w;
    float R_cut, f_R, s_max, s_rs, s_ap;
    float brass_rsp, brass_inv_rsp, brass_rho, brass_inv_X0, brass_za_rho;
    float rs_rsp, rs_inv_rsp, rs_rho, rs_inv_X0, rs_za_rho;
    float rho_min, delta_E;
    float pc2, pc3, pc4, pc5;     // binomial coefficients of (1+d)^p - 1 = d (p + d (pc2 + d (pc3 + ...)))
    int flags;
    double R_cut_d;               // R_cut as fp64: the stop test compares the fp64 range with it every step
};

struct DevGrid {
    int nx, ny, nz;
    float hx, hy, hz;
    float ox, oy, oz;             // low corner
    int hu_min, n_lut;            // material table covers HU in [hu_min, hu_min + n_lut)
};

struct DevBeam {
    float iso[3];
    float rot[9];
    float w_start;                // start plane (depends on scenario when there is no device)
    int has_rs; float w_rs_in, w_rs_out;
    int has_ap; float w_ap_in, w_ap_out;
    const uint32_t *ap_bits;      // row-major, ap_row_words 32-bit words per row, bit ix&31 of word ix>>5
    int ap_nx, ap_ny, ap_row_words;
    float ap_u0, ap_v0, ap_inv_du, ap_inv_dv;    // pixel (ix, iy) = floor((x - u0) / du)
    // safe-distance map of the opening: per tile of kApTile x kApTile pixels, the Chebyshev distance in tiles to the
    // nearest tile that is not fully open (0 = not fully open itself, capped at 255)
    const unsigned char *ap_dist;
    // the same towards the opening: Chebyshev distance in tiles to the nearest tile that holds ANY open pixel
    const unsigned char *ap_dist_open;
    int ap_ntx;
    float ap_tile_u, ap_tile_v;   // tile size in mm
    // S:8f-2: polygon opening (ap_n_poly > 0; no bitmap then).  Vertices (x, y), and a coarse grid over the polygon's bounding
    // box: per cell 0 = the boundary may pass through it (exact test needed), > 0 = wholly inside the opening, < 0 = wholly
    // in brass, |value| = a radius in the L-infinity norm (mm) around ANY point of the cell in which the answer cannot change
    const float2 *ap_poly;
    int ap_n_poly;
    const float *ap_pgrid;
    int ap_pg_nx, ap_pg_ny;
    float ap_pg_x0, ap_pg_y0, ap_pg_inv_cell;
    // per grid row, the edges whose y-range meets the row (+ a rounding margin): the only ones a ray along +x from a point of
    // that row can cross.  ap_prow_ptr [ny + 1], ap_pedges = edge indices (edge k = vertex k -> vertex k + 1)
    const int *ap_prow_ptr;
    const int *ap_pedges;
};

#ifndef VPK_AP_TILE_SHIFT
#define VPK_AP_TILE_SHIFT 0
#endif
constexpr int kApTileShift = VPK_AP_TILE_SHIFT;   // 2^shift x 2^shift pixels per tile of the safe-distance maps

struct Medium { float rsp, inv_rsp, rho_rel, inv_X0, za_rho; };

// One history.  Geometry slots g0..g3: in the beam line they hold the beam-frame lateral position as two fp32 pairs
// (x = g0 + g1, y = g2 + g3, hi + lo) and rz is the LOCAL depth inside the current device; in the CT they hold ix,
// iy, iz and the linear voxel index, and rx, ry, rz are LOCAL offsets inside that voxel (0..h).
struct Hist {
    uint32_t g0, g1, g2, g3;
    float rx, ry, rz;
    float ux, uy, uz;             // direction, high part
    float lx, ly, lz;             // direction, low part (|l| <= ulp(u)/2)
    float E, t_rad, f_rad, tau, tau_star;     // f_rad = 1 + c_log ln t_rad (Highland factor), carried between steps
    double R;                     // residual range in water, alpha E^p
    uint32_t step, hid_lo, hid_hi;
    int region;                   // REG_* | beam index << 8
    int col;                      // influence mode: column (group-local) of this history
};

__device__ __forceinline__ float beam_xh(const Hist &h) { return __uint_as_float(h.g0); }
__device__ __forceinline__ float beam_yh(const Hist &h) { return __uint_as_float(h.g2); }
__device__ __forceinline__ double beam_x(const Hist &h) { return (double)__uint_as_float(h.g0) + (double)__uint_as_float(h.g1); }
__device__ __forceinline__ double beam_y(const Hist &h) { return (double)__uint_as_float(h.g2) + (double)__uint_as_float(h.g3); }
__device__ __forceinline__ void set_beam_x(Hist &h, double x) { const float hi = (float)x; h.g0 = __float_as_uint(hi); h.g1 = __float_as_uint((float)(x - (double)hi)); }
__device__ __forceinline__ void set_beam_y(Hist &h, double y) { const float hi = (float)y; h.g2 = __float_as_uint(hi); h.g3 = __float_as_uint((float)(y - (double)hi)); }

// (hi + lo) += s * (u + l) in fp32 pair arithmetic: exact product by fma, two-sum, renormalise (14 FMA-pipe operations)
__device__ __forceinline__ void pair_axpy(uint32_t &ghi, uint32_t &glo, float s, float u, float l)
{
    const float xh = __uint_as_float(ghi), xl = __uint_as_float(glo);
    const float p = s * u, pe = fmaf(s, u, -p);
    const float S = xh + p, bb = S - xh;
    const float e = (xh - (S - bb)) + (p - bb);
    const float lo = xl + (e + fmaf(s, l, pe));
    const float H = S + lo;
    ghi = __float_as_uint(H); glo = __float_as_uint(lo - (H - S));
}

struct StepOut { float s, dep, removed, theta, uphi; int on_d; };

// fp32 -> fp64 without the flush-to-zero canonicalisation -ftz=true attaches to the plain cast (one FMUL per conversion)
__device__ __forceinline__ double f2d(float x)
{
    double d; asm("cvt.f64.f32 %0, %1;" : "=d"(d) : "f"(x)); return d;
}

// ---------------------------------------------------------------------------------------------- C1
// the ten round keys (k + r * Weyl increment) are the same for every thread: they are computed once on the host and
// sit in the kernel's constant bank, so a round is two wide multiplies and two three-input XORs
struct PhiloxKey { uint32_t k0[10], k1[10]; };

__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, const PhiloxKey &K)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ K.k0[r], n2 = hi0 ^ c3 ^ K.k1[r];
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    }
    return make_uint4(c0, c1, c2, c3);
}

// u = (2*(x>>9)+1) * 2^-24, exact in fp32, strictly inside (0,1).  Built from the bit pattern of 1 + (x>>9) 2^-23
// minus (1 - 2^-24): the subtraction is exact, and no int->float conversion goes through the XU pipe.
__device__ __forceinline__ float u01(uint32_t x)
{
    return __uint_as_float(0x3f800000u | (x >> 9)) - 0.99999994039535522461f;
}

__device__ __forceinline__ float4 draw4(const Hist &h, uint32_t step, uint32_t purpose, const PhiloxKey &K)
{
    const uint4 o = philox4x32_10(h.hid_lo, h.hid_hi, step, purpose, K);
    return make_float4(u01(o.x), u01(o.y), u01(o.z), u01(o.w));
}

// MUFU square root (2 ulp): used where the value is a perturbation, never on the carried state
__device__ __forceinline__ float sqrt_fast(float x)
{
    float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r;
}

// -2 ln u with the MUFU log; guarded against the approximate log crossing zero next to u = 1
__device__ __forceinline__ float bm_radius2_fast(float u)
{
    return fmaxf(-1.3862943611198906f * __log2f(u), 0.0f);
}

// cos / sin of 2 pi u for u in (0,1), argument folded to (-pi, pi) where the MUFU error is 2^-21.4 absolute
__device__ __forceinline__ void sincos_2pi_fast(float u, float *s, float *c)
{
    float sn, cs;
    __sincosf(kTwoPi * (u - 0.5f), &sn, &cs);
    *s = -sn; *c = -cs;
}
__device__ __forceinline__ float cos_2pi_fast(float u) { return -__cosf(kTwoPi * (u - 0.5f)); }

// Highland factor f(t) = 1 + c_log ln t (A(t) = t f(t)^2; f(0) is never used)
__device__ __forceinline__ float highland_f(float t, float c_log) { return t > 0.0f ? fmaf(c_log, __logf(t), 1.0f) : 1.0f; }

// C4-7: A(t + dt) - A(t) without cancellation.  With f' - f = c_log ln(1 + dt/t):
//   A(t') - A(t) = dt f'^2 + t (f' - f)(f' + f).
// f' comes from the MUFU log (absolute error ~6e-9); the DIFFERENCE f' - f is the short series of the log of a ratio
// near 1 when dt/t < 0.1 and the plain difference otherwise (the first steps, where nothing cancels).  Branch-free.
// f_new is returned through `f`.
__device__ __forceinline__ float highland_dA(float t, float dt, float c_log, float &f)
{
    const float tp = t + dt;
    const float fn = highland_f(tp, c_log);
    const float x = __fdividef(dt, fmaxf(t, 1e-30f));
    const float L = x * fmaf(x, fmaf(x, fmaf(x, fmaf(x, fmaf(x, -1.0f / 6.0f, 0.2f), -0.25f), 1.0f / 3.0f), -0.5f), 1.0f);
    const float df = (x < 0.1f) ? c_log * L : fn - f;
    const float dA = (t > 0.0f) ? fmaf(dt, fn * fn, t * df * (fn + f)) : tp * fn * fn;
    f = fn;
    return dA;
}

// ---------------------------------------------------------------------------------------------- C4
// One material step, items 1-7 and 10 (everything but the move and the rotation).  d = geometric limit.  Returns the
// cause; o.theta / o.uphi are the polar deflection and the uniform of the azimuth for rotate().
// Arithmetic organisation (same algorithm as C4, better conditioned in fp32): the oracle carries E and recomputes
// R = alpha E^p every step; in fp32 that round trip loses 2^-24 of the FULL range per step, which the end of range
// amplifies (dE/dR ~ 10 MeV/mm).  Here R is carried in fp64 and updated by differences:
// R' = R - s rsp, and, after straggling, R_next = alpha E'^p = R' (E'/Ebar')^p = R' + R' ((1 + delta)^p - 1).
// FL = the physics switches as a compile-time constant (the kernels are specialised for the default MCS | STRAGGLE | NUCLEAR),
// or -1 = read them from the parameters.
template <int FL>
__device__ __forceinline__ int step_physics(const DevParams &P, Hist &h, const Medium &m, float d,
                                            const PhiloxKey &K, StepOut &o)
{
    const int flags = (FL >= 0) ? FL : P.flags;
    o.removed = 0.0f; o.on_d = 0; o.theta = 0.0f; o.uphi = 0.5f;
    const float E = h.E;
    // 1
    const float R = (float)h.R;
    if (__builtin_expect(h.R <= P.R_cut_d, 0)) { o.dep = E; o.s = 0.0f; h.E = 0.0f; h.R = 0.0; return STOPPED; }
    // 2
    float s = d; int face = 1;
    const float lim = fmaxf(P.f_R * R, P.R_cut) * m.inv_rsp;
    if (lim < s) { s = lim; face = 0; }
    if (P.s_max < s) { s = P.s_max; face = 0; }
    // R' > 0 by construction (C4-2), but inv_rsp is a rounded reciprocal: when the step is the R_cut limit and R is within
    // an ulp of R_cut, s * rsp can exceed R by 1e-7.  R' is kept above 1e-12 mm, so that the logarithm below never sees a
    // non-positive range and the update R_next = R' (E'/Ebar)^p stays what it is everywhere else (R_next <= R_cut then: the
    // history stops at its next step).
    double Rp = fma(-f2d(s), f2d(m.rsp), h.R);
    if (__builtin_expect(__double2hiint(Rp) < 0x3d719799, 0)) Rp = 1e-12;      // Rp < ~1e-12 (or negative): high word below that of 1e-12
    // E is re-derived from the fp64 range every step, so a 3e-7 relative MUFU error does not accumulate
    const float Ebar = exp2f(P.inv_p * __log2f((float)Rp * P.inv_alpha));
    // mean energy lost in the step.  E - Ebar cancels when the step is thin in water-equivalent terms (1 mm of air
    // loses 5e-4 MeV of 150: fp32 resolves 1.5e-5, the MUFU pow 4e-5), so for s rsp / R < 0.03 it is taken from
    // Ebar ((R / R')^(1/p) - 1) = Ebar expm1(-log1p(-x) / p) with two short series (relative error < 1e-7).
    const float x = __fdividef(s * m.rsp, R);
    const float Lm = x * fmaf(x, fmaf(x, fmaf(x, fmaf(x, 0.2f, 0.25f), 1.0f / 3.0f), 0.5f), 1.0f);
    const float y = P.inv_p * Lm;
    const float dEm = (x < 0.03f) ? Ebar * (y * fmaf(y, fmaf(y, fmaf(y, 1.0f / 24.0f, 1.0f / 6.0f), 0.5f), 1.0f)) : E - Ebar;
    // 3
    const float4 u = draw4(h, h.step, 0u, K);
    // 4
    float Ep = Ebar, dep = dEm;
    double Rn = Rp;
    if (flags & 2) {
        const float Emid = 0.5f * (E + Ebar);
        const float g = 1.0f + Emid * (1.0f / kMp);
        const float var = P.k_bohr * m.za_rho * s * 0.5f * fmaf(g, g, 1.0f);   // gamma^2 (1 - beta^2/2) = (gamma^2+1)/2
        const float dE = -sqrt_fast(var * bm_radius2_fast(u.z)) * cos_2pi_fast(u.w);
        Ep = Ebar + dE;
        if (Ep <= 0.0f) { Ep = 0.0f; Rn = 0.0; dep = E; }
        else if (Ep >= E) { Ep = E; Rn = h.R; dep = 0.0f; }
        else {
            dep = dEm - dE;
            const float dl = __fdividef(dE, Ebar);
            float g1;                                   // (1 + dl)^p - 1
            if (fabsf(dl) < 0.05f) g1 = dl * fmaf(dl, fmaf(dl, fmaf(dl, fmaf(dl, P.pc5, P.pc4), P.pc3), P.pc2), P.p);
            else g1 = exp2f(P.p * __log2f(1.0f + dl)) - 1.0f;   // end of range only (sigma_E / E > 5 %): nothing cancels, and a
                                                                // 3e-7 relative error of a residual range of a few mm is 1e-6 mm
            Rn = fma(Rp, f2d(g1), Rp);
        }
    }
    // 5
    o.dep = dep;
    o.s = s;
    // 6
    if (flags & 4) {
        h.tau = fmaf(__fdividef(P.beta_nuc, fmaf(P.beta_nuc, R, 1.0f)) * m.rho_rel, s, h.tau);
        if (__builtin_expect(h.tau >= h.tau_star, 0)) {
            o.dep += P.gamma_loc * Ep;
            o.removed = (1.0f - P.gamma_loc) * Ep;
            h.E = Ep; h.R = Rn;
            return NUCLEAR;
        }
    }
    // 7
    if (flags & 1) {
        const float dt = s * m.inv_X0;
        const float dA = fmaxf(highland_dA(h.t_rad, dt, P.c_log, h.f_rad), 0.0f);
        const float Em = 0.5f * (E + Ep);
        o.theta = __fdividef(P.Es * (Em + kMp), Em * (Em + 2.0f * kMp)) * sqrt_fast(dA * bm_radius2_fast(u.x));
        o.uphi = u.y;
        h.t_rad += dt;
    }
    // 10
    h.E = Ep; h.R = Rn;
    h.step += 1u;
    o.on_d = face;
    return CONT;
}

// C4-8, second half: rotate the direction by (theta, phi = 2 pi uphi).  The direction is the unevaluated sum
// u + l; the rotation is applied as the increment delta = n - u (|delta| ~ theta, so its fp32 rounding is ~1e-9
// absolute) accumulated with an error-free two-sum.  No renormalisation is needed: the increment keeps |u + l| = 1
// to ~1e-9 per step.
__device__ __forceinline__ void rotate(Hist &h, float theta, float uphi)
{
    float sp, cp, st, cm1;
    sincos_2pi_fast(uphi, &sp, &cp);
    if (theta < 0.25f) {        // Taylor to theta^7 / theta^8: error < 2e-9
        const float t2 = theta * theta;
        st = theta * fmaf(t2, fmaf(t2, fmaf(t2, -1.0f / 5040.0f, 1.0f / 120.0f), -1.0f / 6.0f), 1.0f);
        cm1 = t2 * fmaf(t2, fmaf(t2, fmaf(t2, 1.0f / 40320.0f, -1.0f / 720.0f), 1.0f / 24.0f), -0.5f);
    } else {
        float ct;                  // rare (end of range): MUFU accuracy (2^-21 absolute) is enough here
        __sincosf(theta, &st, &ct);
        cm1 = ct - 1.0f;
    }
    const float ux = h.ux, uy = h.uy, uw = h.uz;
    const float rho2 = fmaf(ux, ux, uy * uy);
    float dx, dy, dw;
    if (rho2 < 1e-10f) {
        const float sg = (uw < 0.0f) ? -1.0f : 1.0f;
        dx = fmaf(st, cp, -ux); dy = fmaf(st, sp, -uy); dw = fmaf(sg, cm1, sg - uw);
    } else {
        const float isq = rsqrtf(rho2);
        const float a = st * isq;
        dx = fmaf(ux, cm1, a * fmaf(ux * uw, cp, -uy * sp));
        dy = fmaf(uy, cm1, a * fmaf(uy * uw, cp, ux * sp));
        dw = fmaf(uw, cm1, -(rho2 * isq) * st * cp);
    }
    // two-sum accumulate, then re-split so that |l| <= ulp(u)/2
#define VPK_ACC(U, L, D)                                                  \
    {                                                                     \
        const float S = U + D, bb = S - U;                                \
        const float e = (U - (S - bb)) + (D - bb);                        \
        const float l2 = L + e, S2 = S + l2;                              \
        L = l2 - (S2 - S); U = S2;                                        \
    }
    VPK_ACC(h.ux, h.lx, dx)
    VPK_ACC(h.uy, h.ly, dy)
    VPK_ACC(h.uz, h.lz, dw)
#undef VPK_ACC
}

}  // namespace vpk
