// vpmc_influence.inl -- S7/S8: per-(scenario, spot) columns and the CSR writer (included by vpmc_run.inl).

extern "C" int vpmc_influence(vpmc_t *h, const vpmc_scenario *sc, int32_t n_sc, uint32_t hist_per_spot,
                              float rel_threshold, uint64_t seed, vpmc_csr *out, vpmc_alloc_fn alloc, void *user,
                              void *cuda_stream)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    (void)sc; (void)n_sc; (void)hist_per_spot; (void)rel_threshold; (void)seed; (void)out; (void)alloc; (void)user; (void)cuda_stream;
    FAIL(h, VPMC_ERR_STATE, "vpmc_influence: not built yet");
}

extern "C" int vpmc_csr_from_dense(vpmc_t *h, const float *col_dev, int64_t n, float rel_threshold,
                                   int32_t *col_out_dev, float *val_out_dev, int64_t *nnz_out)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    (void)col_dev; (void)n; (void)rel_threshold; (void)col_out_dev; (void)val_out_dev; (void)nnz_out;
    FAIL(h, VPMC_ERR_STATE, "vpmc_csr_from_dense: not built yet");
}
