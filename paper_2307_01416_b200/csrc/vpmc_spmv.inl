// vpmc_spmv.inl -- host side of SURVEY.md 8(f)-1 (included by vpmc_run.inl): launches of vpmc_spmv.cuh.

static int check_csr(vpmc_t *h, const vpmc_csr *m)
{
    if (!m || !m->row_ptr || m->n_rows < 0 || m->nnz < 0 || (m->nnz > 0 && (!m->col || !m->val))) FAIL(h, VPMC_ERR_INVALID_ARG, "bad CSR matrix");
    return VPMC_OK;
}

static int spmv_chunks(long long nnz) { return (int)((nnz + kSpmvChunk - 1) / kSpmvChunk); }

static int spmv_dose_launch(vpmc_t *h, const vpmc_csr *m, int64_t n_cols, const float *w, float *d, cudaStream_t st)
{
    CU(h, cudaMemsetAsync(d, 0, (size_t)n_cols * sizeof(float), st));
    if (m->nnz > 0) {
        spmv_dose_kernel<<<spmv_chunks(m->nnz), kSpmvBlock, 0, st>>>((const long long *)m->row_ptr, m->col, m->val, m->n_rows, m->nnz, w, d);
        CU(h, cudaGetLastError());
        h->launches += 1;
    }
    return VPMC_OK;
}

static int spmv_grad_launch(vpmc_t *h, const vpmc_csr *m, const float *r, float *g, int accumulate, cudaStream_t st)
{
    const int nc = spmv_chunks(m->nnz);
    int rc = ensure(h, h->spmv_part, (size_t)std::max(nc, 1) * 2 * sizeof(float)); if (rc) return rc;
    float *fp = h->spmv_part.as<float>(), *lp = fp + std::max(nc, 1);
    if (nc > 0) {
        spmv_grad_kernel<<<nc, kSpmvBlock, 0, st>>>((const long long *)m->row_ptr, m->col, m->val, m->n_rows, m->nnz, r, g, accumulate, fp, lp);
        h->launches += 1;
    }
    if (m->n_rows > 0) {
        spmv_grad_fixup_kernel<<<(m->n_rows + 255) / 256, 256, 0, st>>>((const long long *)m->row_ptr, m->n_rows, fp, lp, g, accumulate);
        h->launches += 1;
    }
    CU(h, cudaGetLastError());
    return VPMC_OK;
}

extern "C" int vpmc_spmv_dose(vpmc_t *h, const vpmc_csr *m, int64_t n_cols, const float *w_dev, float *dose_dev, void *cuda_stream)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    int rc = check_csr(h, m); if (rc) return rc;
    if (n_cols < 1 || !dose_dev || (m->n_rows > 0 && !w_dev)) FAIL(h, VPMC_ERR_INVALID_ARG, "bad spmv_dose arguments");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    h->last_stream = st; h->launched = true;
    TimedScope ts(h, st, 5);
    return spmv_dose_launch(h, m, n_cols, w_dev, dose_dev, st);
}

extern "C" int vpmc_spmv_grad(vpmc_t *h, const vpmc_csr *m, const float *r_dev, float *grad_dev, int accumulate, void *cuda_stream)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    int rc = check_csr(h, m); if (rc) return rc;
    if ((m->n_rows > 0 && !grad_dev) || (m->nnz > 0 && !r_dev)) FAIL(h, VPMC_ERR_INVALID_ARG, "bad spmv_grad arguments");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    h->last_stream = st; h->launched = true;
    TimedScope ts(h, st, 5);
    return spmv_grad_launch(h, m, r_dev, grad_dev, accumulate, st);
}

extern "C" int vpmc_worst_case(vpmc_t *h, const float *doses_dev, int32_t n_sc, int64_t n, const float *target_dev, const float *weight_dev,
                               float *resid_dev, double *objective_dev, void *cuda_stream)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    if (!doses_dev || n_sc < 1 || n < 1 || !target_dev || !weight_dev || !resid_dev || !objective_dev) FAIL(h, VPMC_ERR_INVALID_ARG, "bad worst_case arguments");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    h->last_stream = st; h->launched = true;
    TimedScope ts(h, st, 5);
    CU(h, cudaMemsetAsync(objective_dev, 0, sizeof(double), st));
    worst_case_kernel<<<grid_for(n, h->n_sm), 256, 0, st>>>(doses_dev, n_sc, n, target_dev, weight_dev, resid_dev, objective_dev);
    CU(h, cudaGetLastError());
    h->launches += 1;
    return VPMC_OK;
}

extern "C" int vpmc_robust_iteration(vpmc_t *h, const vpmc_csr *mats, int32_t n_sc, int64_t n_cols, const float *w_dev, const float *target_dev,
                                     const float *weight_dev, float *doses_ws_dev, float *resid_ws_dev, float *grad_dev, double *objective_dev,
                                     void *cuda_stream)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    if (!mats || n_sc < 1 || n_cols < 1 || !w_dev || !target_dev || !weight_dev || !doses_ws_dev || !resid_ws_dev || !grad_dev || !objective_dev)
        FAIL(h, VPMC_ERR_INVALID_ARG, "bad robust_iteration arguments");
    for (int s = 0; s < n_sc; ++s) {
        int rc = check_csr(h, mats + s); if (rc) return rc;
        if (mats[s].n_rows != mats[0].n_rows) FAIL(h, VPMC_ERR_INVALID_ARG, "scenario %d has %d rows, scenario 0 has %d", s, mats[s].n_rows, mats[0].n_rows);
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    h->last_stream = st; h->launched = true;
    TimedScope ts(h, st, 5);
    int rc;
    for (int s = 0; s < n_sc; ++s)
        if ((rc = spmv_dose_launch(h, mats + s, n_cols, w_dev, doses_ws_dev + (size_t)s * n_cols, st))) return rc;
    CU(h, cudaMemsetAsync(objective_dev, 0, sizeof(double), st));
    worst_case_kernel<<<grid_for(n_cols, h->n_sm), 256, 0, st>>>(doses_ws_dev, n_sc, n_cols, target_dev, weight_dev, resid_ws_dev, objective_dev);
    CU(h, cudaGetLastError());
    h->launches += 1;
    for (int s = 0; s < n_sc; ++s)        // the scenarios' gradients are added in scenario order
        if ((rc = spmv_grad_launch(h, mats + s, resid_ws_dev + (size_t)s * n_cols, grad_dev, s > 0, st))) return rc;
    return VPMC_OK;
}

// ---- S:8f-3: 3-D gamma index of two dose grids of this engine's CT (vpmc_gamma.cuh)
extern "C" int vpmc_gamma(vpmc_t *h, const float *ref_dev, const float *eval_dev, float dd_rel, float dta_mm, float threshold_rel, int32_t sub,
                          uint64_t *n_eval_out, uint64_t *n_fail_out, void *cuda_stream)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    if (!ref_dev || !eval_dev || !(dd_rel > 0) || !(dta_mm > 0) || !(threshold_rel >= 0) || sub < 1 || sub > 64 || !n_eval_out || !n_fail_out)
        FAIL(h, VPMC_ERR_INVALID_ARG, "bad gamma arguments");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    h->last_stream = st; h->launched = true;
    int rc;
    const unsigned int cap = (unsigned int)std::min<long long>(h->ncell, 0x7fffffffLL);
    if ((rc = ensure(h, h->gamma_buf, sizeof(GammaCounts) + (size_t)cap * sizeof(unsigned int)))) return rc;
    GammaCounts *c = h->gamma_buf.as<GammaCounts>();
    unsigned int *list = reinterpret_cast<unsigned int *>(c + 1);
    // the grids are on the scoring grid: cells of sdiv voxels per axis
    GammaArgs a = { h->sn[0], h->sn[1], h->sn[2], h->G.hx * (float)h->sdiv[0], h->G.hy * (float)h->sdiv[1], h->G.hz * (float)h->sdiv[2], dd_rel, dta_mm,
                    threshold_rel, (int)sub };
    CU(h, cudaMemsetAsync(c, 0, sizeof(GammaCounts), st));
    const int g = grid_for(h->ncell, h->n_sm);
    gamma_max_kernel<<<g, 256, 0, st>>>(ref_dev, h->ncell, c);
    gamma_select_kernel<<<g, 256, 0, st>>>(ref_dev, eval_dev, h->ncell, a, c, list, cap);
    gamma_search_kernel<<<h->n_sm * 8, 256, 0, st>>>(ref_dev, eval_dev, a, c, list, cap);
    CU(h, cudaGetLastError());
    h->launches += 3;
    GammaCounts out;
    CU(h, cudaMemcpyAsync(&out, c, sizeof(out), cudaMemcpyDeviceToHost, st));
    CU(h, cudaStreamSynchronize(st));
    *n_eval_out = out.n_eval; *n_fail_out = out.n_fail;
    return VPMC_OK;
}
