/*
 * robust_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain CPU oracle of one iteration of the robust optimiser on the influence matrices the transport path writes
 * ("0.1-0.3 s per iteration", "13 uncertainty scenarios were included in the robust
 * optimization", "on-the-fly optimization ... 71.4 seconds").  The paper gives no formula for its objective; the
 * reading taken (R16) is the voxel-wise worst case over the scenarios of a weighted quadratic deviation:
 *
 *   d_s[v]  = sum_j D_s[j][v] w_j                                   dose of scenario s (D_s: rows = spots j, CSR, C6)
 *   e_s[v]  = d_s[v] - t[v]
 *   s*(v)   = the scenario with the largest e_s[v]^2, the lowest index among equals; this one comparison is taken in fp32
 *             (difference and product each rounded to fp32), the precision the kernel takes it in, so that both sides
 *             decide the integer s* alike on fp32 inputs; every value (f, r, g) is fp64
 *   f(w)    = sum_v p[v] e_{s*(v)}[v]^2
 *   r_s[v]  = 2 p[v] e_s[v] if s = s*(v), else 0
 *   g[j]    = sum_s sum_v D_s[j][v] r_s[v]                           gradient of f where s* is locally constant
 *
 * Written as the definitions: nested loops, fp64 accumulation, no blocking.  Shares nothing with the CUDA path.
 * Pins (tests/test_oracle_robust.py): dense numpy products on small matrices, the adjoint identity <D w, r> = <w, D^T r>,
 * a central finite difference of f against g, hand-computed 2-voxel cases.
 */
#include <stdint.h>
#include <stddef.h>

/* d[v] = sum_j D[j][v] w[j]; d has n_cols entries and is overwritten */
void orb_spmv_dose(const int64_t *row_ptr, const int32_t *col, const float *val, int32_t n_rows, int64_t n_cols,
                   const double *w, double *d)
{
    for (int64_t v = 0; v < n_cols; ++v) d[v] = 0.0;
    for (int32_t j = 0; j < n_rows; ++j)
        for (int64_t k = row_ptr[j]; k < row_ptr[j + 1]; ++k) d[col[k]] += (double)val[k] * w[j];
}

/* g[j] (+)= sum_v D[j][v] r[v] */
void orb_spmv_grad(const int64_t *row_ptr, const int32_t *col, const float *val, int32_t n_rows, const double *r,
                   int32_t accumulate, double *g)
{
    for (int32_t j = 0; j < n_rows; ++j) {
        double s = 0.0;
        for (int64_t k = row_ptr[j]; k < row_ptr[j + 1]; ++k) s += (double)val[k] * r[col[k]];
        g[j] = accumulate ? g[j] + s : s;
    }
}

/* doses, resid: [n_sc][n] row-major.  Returns f; resid is overwritten; worst[v] (may be NULL) = s*(v) */
double orb_worst_case(const double *doses, int32_t n_sc, int64_t n, const double *target, const double *weight,
                      double *resid, int32_t *worst)
{
    double f = 0.0;
    for (int64_t v = 0; v < n; ++v) {
        int32_t best = 0;
        double e_best = doses[v] - target[v];
        volatile float q_best = (float)doses[v] - (float)target[v];
        q_best = q_best * q_best;
        for (int32_t s = 1; s < n_sc; ++s) {
            const double e = doses[(size_t)s * n + v] - target[v];
            volatile float q = (float)doses[(size_t)s * n + v] - (float)target[v];
            q = q * q;
            if (q > q_best) { e_best = e; best = s; q_best = q; }
        }
        for (int32_t s = 0; s < n_sc; ++s) resid[(size_t)s * n + v] = 0.0;
        resid[(size_t)best * n + v] = 2.0 * weight[v] * e_best;
        f += weight[v] * e_best * e_best;
        if (worst) worst[v] = best;
    }
    return f;
}
