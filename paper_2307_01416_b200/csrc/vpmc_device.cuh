// vpmc_device.cuh -- device-side transport primitives (fp32) shared by the beam-line kernel, the voxel
// kernel and the trace kernel.  Written for sm_100a.  Independent of oracle/ (no shared code or tables).
//
// Physics: SURVEY.md 8(c) C1-C5 (closed-form reading of P:L73-P:L87).  Precision plan:
// the carried state chain E -> R -> R' -> E' uses accurate powf; the random deviates (Box-Muller, azimuth)
// use MUFU-based fast intrinsics because they enter only as small perturbations of the state.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace vpk {

constexpr float kMp = 938.272f;
constexpr float kTwoPi = 6.283185307179586f;

enum : int { REG_VAC = 0, REG_RS = 1, REG_AP_OPEN = 2, REG_AP_BRASS = 3, REG_CT = 4 };
enum : int { CONT = 0, STOPPED = 1, NUCLEAR = 2, ESCAPED = 3 };

// Parameters in device form (constant memory).
struct DevParams {
    float alpha, p, inv_p, inv_alpha;
    float inv_X0_w, Es, c_log;
    float beta_nuc, gamma_loc, k_bohr, za_w;
    float R_cut, f_R, s_max, s_rs, s_ap;
    float brass_rsp, brass_rho, brass_inv_X0, brass_za_rho;
    float rs_rsp, rs_rho, rs_inv_X0, rs_za_rho;
    float rho_min, delta_E;
    float pc2, pc3, pc4, pc5;     // binomial coefficients of (1+d)^p - 1 = d (p + d (pc2 + d (pc3 + ...)))
    int flags;
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
    float ap_u0, ap_v0, ap_du, ap_dv;
};

struct Medium { float rsp, rho_rel, inv_X0, za_rho; };

// Position variables: in a beam-line device rx, ry are beam-frame x, y and rz is the LOCAL depth inside the
// device; in the CT rx, ry, rz are LOCAL offsets inside the current voxel (0..h).  Local coordinates keep the
// fp32 rounding of a position at 1e-7 mm instead of 1e-5 mm.  R is the residual range in water,
// alpha E^p, carried in fp64: it is the well-conditioned state variable; E is re-derived from it every step.
struct Hist {
    float rx, ry, rz, ux, uy, uz;
    float E, t_rad, A_rad, tau, tau_star;     // A_rad = highland_A(t_rad), carried to save a log per step
    double R;
    uint32_t step, hid_lo, hid_hi;
};

struct StepOut { float s, dep, removed; int on_d; };

// ---------------------------------------------------------------------------------------------- C1
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return make_uint4(c0, c1, c2, c3);
}

// u = (2*(x>>9)+1) * 2^-24, exact in fp32, strictly inside (0,1)
__device__ __forceinline__ float u01(uint32_t x)
{
    return __uint2float_rn(2u * (x >> 9) + 1u) * 5.9604644775390625e-8f;
}

__device__ __forceinline__ float4 draw4(const Hist &h, uint32_t step, uint32_t purpose, uint32_t k0, uint32_t k1)
{
    const uint4 o = philox4x32_10(h.hid_lo, h.hid_hi, step, purpose, k0, k1);
    return make_float4(u01(o.x), u01(o.y), u01(o.z), u01(o.w));
}

// MUFU square root (2 ulp): used where the value is a perturbation, never on the carried state
__device__ __forceinline__ float sqrt_fast(float x)
{
    float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r;
}

// sqrt(-2 ln u) with the MUFU log; guarded against the approximate log crossing zero next to u = 1
__device__ __forceinline__ float bm_radius_fast(float u)
{
    return sqrt_fast(fmaxf(-1.3862943611198906f * __log2f(u), 0.0f));
}

// cos / sin of 2 pi u for u in (0,1), argument folded to (-pi, pi) where the MUFU error is 2^-21.4 absolute
__device__ __forceinline__ void sincos_2pi_fast(float u, float *s, float *c)
{
    float sn, cs;
    __sincosf(kTwoPi * (u - 0.5f), &sn, &cs);
    *s = -sn; *c = -cs;
}

__device__ __forceinline__ float highland_A(float t, float c_log)
{
    if (t <= 0.0f) return 0.0f;
    const float f = fmaf(c_log, __logf(t), 1.0f);
    return t * f * f;
}

// ---------------------------------------------------------------------------------------------- C4
// One material step, items 1-8 and 10.  d = geometric limit.  Returns the cause.
// Arithmetic organisation (same algorithm as C4, better conditioned in fp32): the oracle carries E and
// recomputes R = alpha E^p every step; in fp32 that round trip loses 2^-24 of the FULL range per step, which the
// end of range amplifies (dE/dR ~ 10 MeV/mm).  Here R is carried in fp64 and updated by differences:
// R' = R - s rsp, and, after straggling, R_next = alpha E'^p = R' (E'/Ebar')^p = R' + R' expm1(p log1p(delta)).
__device__ __forceinline__ int material_step(const DevParams &P, Hist &h, const Medium &m, float d,
                                             uint32_t k0, uint32_t k1, StepOut &o)
{
    o.removed = 0.0f; o.on_d = 0;
    const float E = h.E;
    // 1
    const float R = (float)h.R;
    if (h.R <= (double)P.R_cut) { o.dep = E; o.s = 0.0f; h.E = 0.0f; h.R = 0.0; return STOPPED; }
    // 2
    float s = d; int face = 1;
    const float lim = __fdividef(fmaxf(P.f_R * R, P.R_cut), m.rsp);
    if (lim < s) { s = lim; face = 0; }
    if (P.s_max < s) { s = P.s_max; face = 0; }
    const double Rp = fma(-(double)s, (double)m.rsp, h.R);
    // E is re-derived from the fp64 range every step, so a 3e-7 relative MUFU error does not accumulate
    const float Ebar = exp2f(P.inv_p * __log2f((float)Rp * P.inv_alpha));
    // 3
    const float4 u = draw4(h, h.step, 0u, k0, k1);
    // 4
    float Ep = Ebar;
    double Rn = Rp;
    if (P.flags & 2) {
        const float Emid = 0.5f * (E + Ebar);
        const float g = 1.0f + Emid * (1.0f / kMp);
        const float var = P.k_bohr * m.za_rho * s * 0.5f * fmaf(g, g, 1.0f);   // gamma^2 (1 - beta^2/2) = (gamma^2+1)/2
        float sn, cs;
        sincos_2pi_fast(u.w, &sn, &cs);
        const float dE = -sqrt_fast(var) * (bm_radius_fast(u.z) * cs);
        Ep = Ebar + dE;
        if (Ep <= 0.0f) { Ep = 0.0f; Rn = 0.0; }
        else if (Ep >= E) { Ep = E; Rn = h.R; }
        else {
            const float dl = __fdividef(dE, Ebar);
            float g1;                                   // (1 + dl)^p - 1
            if (fabsf(dl) < 0.05f) g1 = dl * fmaf(dl, fmaf(dl, fmaf(dl, fmaf(dl, P.pc5, P.pc4), P.pc3), P.pc2), P.p);
            else g1 = expm1f(P.p * log1pf(dl));
            Rn = fma(Rp, (double)g1, Rp);
        }
    }
    // 5
    o.dep = E - Ep;
    o.s = s;
    // 6
    if (P.flags & 4) {
        h.tau = fmaf(__fdividef(P.beta_nuc, fmaf(P.beta_nuc, R, 1.0f)) * m.rho_rel, s, h.tau);
        if (h.tau >= h.tau_star) {
            o.dep += P.gamma_loc * Ep;
            o.removed = (1.0f - P.gamma_loc) * Ep;
            h.E = Ep; h.R = Rn;
            return NUCLEAR;
        }
    }
    // 7
    float theta = 0.0f, sp = 0.0f, cp = 1.0f;
    if (P.flags & 1) {
        const float tp = fmaf(s, m.inv_X0, h.t_rad);
        const float Ap = highland_A(tp, P.c_log);
        const float dA = fmaxf(Ap - h.A_rad, 0.0f);
        const float Em = 0.5f * (E + Ep);
        theta = __fdividef(P.Es * (Em + kMp), Em * (Em + 2.0f * kMp)) * sqrt_fast(dA) * bm_radius_fast(u.x);
        sincos_2pi_fast(u.y, &sp, &cp);
        h.t_rad = tp; h.A_rad = Ap;
    }
    // 8: move along the old direction, then rotate about it
    h.rx = fmaf(s, h.ux, h.rx); h.ry = fmaf(s, h.uy, h.ry); h.rz = fmaf(s, h.uz, h.rz);
    if (P.flags & 1) {
        float st, ct;
        if (theta < 0.25f) {        // Taylor to theta^7 / theta^8: error < 2e-9
            const float t2 = theta * theta;
            st = theta * fmaf(t2, fmaf(t2, fmaf(t2, -1.0f / 5040.0f, 1.0f / 120.0f), -1.0f / 6.0f), 1.0f);
            ct = fmaf(t2, fmaf(t2, fmaf(t2, fmaf(t2, 1.0f / 40320.0f, -1.0f / 720.0f), 1.0f / 24.0f), -0.5f), 1.0f);
        } else {
            sincosf(theta, &st, &ct);
        }
        const float ux = h.ux, uy = h.uy, uw = h.uz;
        const float rho2 = fmaf(ux, ux, uy * uy);
        float nx, ny, nw;
        if (rho2 < 1e-10f) {
            nx = st * cp; ny = st * sp; nw = (uw < 0.0f) ? -ct : ct;
        } else {
            const float isq = rsqrtf(rho2);
            const float a = st * isq;
            nx = fmaf(ux, ct, a * fmaf(ux * uw, cp, -uy * sp));
            ny = fmaf(uy, ct, a * fmaf(uy * uw, cp, ux * sp));
            nw = fmaf(uw, ct, -(rho2 * isq) * st * cp);
        }
        const float inrm = rsqrtf(fmaf(nx, nx, fmaf(ny, ny, nw * nw)));
        h.ux = nx * inrm; h.uy = ny * inrm; h.uz = nw * inrm;
    }
    // 10
    h.E = Ep; h.R = Rn;
    h.step += 1u;
    o.on_d = face;
    return CONT;
}

}  // namespace vpk
