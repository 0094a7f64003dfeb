// vpmc_influence.inl -- S7/S8: per-(scenario, spot) columns and the CSR writer (included by vpmc_run.inl).
//
// Per scenario:
//   1. pilot: the first n_pilot histories of every spot run in MODE 2 and leave the bounding box of their deposits;
//   2. boxes: the pilot box of each column, grown by box_grow of its extent + box_pad voxels per side, clipped to the grid
//      (tight on purpose: the overflow list of step 4 takes the halo, and every box element is zeroed and scanned);
//   3. columns are packed into groups whose boxes fit the workspace; per group: zero the boxes, transport all
//      hist_per_spot histories of the group's spots in MODE 1, then max / count / scan / emit into a staging area;
//   4. deposits outside a column's box go to an overflow list of (column, voxel, MeV) entries, which is bucketed by column,
//      sorted by voxel and summed per voxel by one CTA per column, thresholded with the column and merged into the row at
//      the end.  Only when that list is full (or a column's bucket exceeds what a CTA sorts) is a column NOT written: its box is replaced by the union with the bounding box of the lost deposits and the column is
//      replayed in a later group -- streams are keyed by history id, so the replay reproduces the same histories and
//      now fits by construction;
//   5. row_ptr = exclusive scan of the row counts; the caller's allocator provides row_ptr / col / val and the rows are
//      gathered from the staging area.

struct HostBox { int lo[3], dim[3]; long long vol() const { return (long long)dim[0] * dim[1] * dim[2]; } };

template <class T>
static int upload(vpmc_t *h, DevBuf &b, const std::vector<T> &v, cudaStream_t st)
{
    int rc = ensure(h, b, std::max<size_t>(v.size(), 1) * sizeof(T)); if (rc) return rc;
    if (!v.empty()) CU(h, cudaMemcpyAsync(b.p, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice, st));
    return VPMC_OK;
}

// grow a device buffer keeping its first `keep` bytes
static int grow_keep(vpmc_t *h, DevBuf &b, size_t bytes, size_t keep, cudaStream_t st)
{
    if (b.bytes >= bytes && b.p) return VPMC_OK;
    void *np = nullptr;
    const size_t want = std::max(bytes, b.bytes + b.bytes / 2);
    if (cudaMalloc(&np, want) != cudaSuccess) { cudaGetLastError(); FAIL(h, VPMC_ERR_ALLOC, "out of device memory (%zu bytes of CSR staging)", want); }
    if (b.p && keep) CU(h, cudaMemcpyAsync(np, b.p, keep, cudaMemcpyDeviceToDevice, st));
    CU(h, cudaStreamSynchronize(st));
    if (b.p) pool_give(b.p, b.bytes);       // the stream was synchronised just above
    b.p = np; b.bytes = want;
    return VPMC_OK;
}

// grid of a writer pass that strides over the tiles: all CTAs resident at once (n_sm x the kernel's own occupancy, looked up
// once) -- with a fixed 8 per SM the 40-register conversion pass ran 1.33 waves, its last third on a third of the machine
static int tile_grid(vpmc_t *h, const void *kernel, int n_tiles)
{
    static std::mutex mu;
    static std::vector<std::pair<const void *, int>> cache;      // per kernel; every device here is the same part
    int occ = 0;
    {
        std::lock_guard<std::mutex> lk(mu);
        for (auto &e : cache) if (e.first == kernel) occ = e.second;
        if (occ == 0) {
            if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, kBlock, 0) != cudaSuccess || occ < 1) { cudaGetLastError(); occ = 4; }
            cache.push_back({ kernel, occ });
        }
    }
    return std::max(1, std::min(n_tiles, h->n_sm * occ));
}

// writer pass 1 over a set of columns: (E_dep -> dose value,) column maxima
static int csr_max_pass(vpmc_t *h, const CsrCols &cc, float *data, bool convert, float coef, cudaStream_t st)
{
    int rc = ensure(h, h->inf_colmax, (size_t)cc.n_cols * sizeof(unsigned int)); if (rc) return rc;
    CU(h, cudaMemsetAsync(h->inf_colmax.p, 0, (size_t)cc.n_cols * sizeof(unsigned int), st));
    if (cc.n_tiles > 0) {
        const int grid = convert ? tile_grid(h, (const void *)csr_max_kernel<true>, cc.n_tiles) : tile_grid(h, (const void *)csr_max_kernel<false>, cc.n_tiles);
        TimedScope ts(h, st, 3);
        if (convert)
            csr_max_kernel<true><<<grid, kBlock, 0, st>>>(cc, data, h->d_hu, h->d_lut, h->G.hu_min, h->G.n_lut, h->params.rho_min, coef, h->inf_colmax.as<unsigned int>(), h->d_cell_rho);
        else
            csr_max_kernel<false><<<grid, kBlock, 0, st>>>(cc, data, h->d_hu, h->d_lut, h->G.hu_min, h->G.n_lut, h->params.rho_min, coef, h->inf_colmax.as<unsigned int>(), nullptr);
        CU(h, cudaGetLastError());
        h->launches += 1;
    }
    return VPMC_OK;
}

// writer passes 2 + 3: kept entries per tile, exclusive scan per column; leaves per-column counts in inf_colnnz (device)
static int csr_count_pass(vpmc_t *h, const CsrCols &cc, const float *data, float rel_thr, cudaStream_t st)
{
    int rc = ensure(h, h->inf_tilecnt, (size_t)std::max(cc.n_tiles, 1) * sizeof(unsigned int)); if (rc) return rc;
    rc = ensure(h, h->inf_colnnz, (size_t)cc.n_cols * sizeof(long long)); if (rc) return rc;
    TimedScope ts(h, st, 3);
    if (cc.n_tiles > 0) {
        csr_count_kernel<<<tile_grid(h, (const void *)csr_count_kernel, cc.n_tiles), kBlock, 0, st>>>(cc, data, h->inf_colmax.as<unsigned int>(), rel_thr, h->inf_tilecnt.as<unsigned int>());
        h->launches += 1;
    }
    csr_tile_scan_kernel<<<cc.n_cols, kBlock, 0, st>>>(cc, h->inf_tilecnt.as<unsigned int>(), h->inf_colnnz.as<long long>());
    CU(h, cudaGetLastError());
    h->launches += 1;
    return VPMC_OK;
}

extern "C" int vpmc_csr_from_dense(vpmc_t *h, const float *col_dev, int64_t n, float rel_threshold,
                                   int32_t *col_out_dev, float *val_out_dev, int64_t *nnz_out)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    if (!col_dev || n < 0 || n > 0x7fffffffLL || !nnz_out || (!col_out_dev) != (!val_out_dev)) FAIL(h, VPMC_ERR_INVALID_ARG, "bad csr_from_dense arguments");
    *nnz_out = 0;
    if (n == 0) return VPMC_OK;
    cudaStream_t st = nullptr;
    std::vector<int4> lo(1, make_int4(0, 0, 0, 0)), dim(1, make_int4((int)n, 1, 1, 0));
    std::vector<unsigned long long> off(1, 0ull);
    std::vector<int> tile0 = { 0, (int)((n + kTile - 1) / kTile) };
    int rc;
    if ((rc = upload(h, h->inf_lo, lo, st)) || (rc = upload(h, h->inf_dim, dim, st)) || (rc = upload(h, h->inf_off, off, st)) ||
        (rc = upload(h, h->inf_tile0, tile0, st))) return rc;
    CsrCols cc{};
    cc.lo = h->inf_lo.as<int4>(); cc.dim = h->inf_dim.as<int4>(); cc.offset = h->inf_off.as<unsigned long long>();
    cc.tile0 = h->inf_tile0.as<int>(); cc.skip = nullptr; cc.n_cols = 1; cc.n_tiles = tile0[1]; cc.nx = (int)n; cc.ny = 1;
    rc = csr_max_pass(h, cc, const_cast<float *>(col_dev), false, 1.0f, st); if (rc) return rc;
    rc = csr_count_pass(h, cc, col_dev, rel_threshold, st); if (rc) return rc;
    long long nnz = 0;
    CU(h, cudaMemcpy(&nnz, h->inf_colnnz.p, sizeof(long long), cudaMemcpyDeviceToHost));
    *nnz_out = nnz;
    if (col_out_dev && nnz > 0) {
        std::vector<long long> base(1, 0ll);
        rc = upload(h, h->inf_colbase, base, st); if (rc) return rc;
        csr_emit_kernel<<<tile_grid(h, (const void *)csr_emit_kernel, cc.n_tiles), kBlock, 0, st>>>(cc, col_dev, h->inf_colmax.as<unsigned int>(), rel_threshold,
                                                                                         h->inf_tilecnt.as<unsigned int>(), h->inf_colbase.as<long long>(), col_out_dev, val_out_dev);
        CU(h, cudaGetLastError());
        h->launches += 1;
        CU(h, cudaStreamSynchronize(st));
    }
    return VPMC_OK;
}

extern "C" int vpmc_get_influence_stats(vpmc_t *h, vpmc_influence_stats *out)
{
    if (!h || !out) return VPMC_ERR_INVALID_ARG;
    *out = h->inf_stats;
    return VPMC_OK;
}

extern "C" int vpmc_set_workspace_limit(vpmc_t *h, uint64_t bytes)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    h->workspace_limit = (size_t)bytes;
    return VPMC_OK;
}

static HostBox grown_box(const int bb[6], const int n[3], float grow, int pad_vox)
{
    HostBox b;
    for (int a = 0; a < 3; ++a) {
        const int ext = bb[3 + a] - bb[a] + 1;
        const int pad = (int)std::ceil(grow * (float)ext) + pad_vox;
        const int lo = std::max(bb[a] - pad, 0), hi = std::min(bb[3 + a] + pad, n[a] - 1);
        b.lo[a] = lo; b.dim[a] = hi - lo + 1;
    }
    return b;
}

extern "C" int vpmc_influence(vpmc_t *h, const vpmc_scenario *scs, int32_t n_sc, uint32_t hist_per_spot,
                              float rel_threshold, uint64_t seed, vpmc_csr *out, vpmc_alloc_fn alloc, void *user,
                              void *cuda_stream)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    if (!scs || n_sc < 1 || hist_per_spot < 1 || !out || !alloc || !(rel_threshold >= 0.0f)) FAIL(h, VPMC_ERR_INVALID_ARG, "bad influence arguments");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    h->last_stream = st;
    h->unc_valid = false;
    for (int s = 0; s < n_sc; ++s) { out[s].row_ptr = nullptr; out[s].col = nullptr; out[s].val = nullptr; out[s].nnz = 0; out[s].n_rows = 0; }
    CU(h, cudaMemsetAsync(h->d_tal, 0, sizeof(DevTallies), st));
    h->inf_stats = vpmc_influence_stats{};
    size_t limit = h->workspace_limit;
    if (limit == 0) {
        size_t fr = 0, tot = 0;
        CU(h, cudaMemGetInfo(&fr, &tot));
        limit = std::min<size_t>((size_t)24 << 30, fr / 3);
    }
    const long long limit_elems = std::max<long long>((long long)(limit / sizeof(float)), 1);
    const double V = (double)h->G.hx * h->G.hy * h->G.hz * 1e-3;
    const float coef = (float)(1.0 / (double)hist_per_spot / V * 1.602176634e-10);          // C6: scale 1 / hist_per_spot
    const uint32_t n_pilot = std::min<uint32_t>(hist_per_spot, std::max<uint32_t>(32u, hist_per_spot / 32u));
    const unsigned int ovf_cap = h->ovf_cap;  // entries of the overflow list (12 B each); 0 forces replays

    for (int s = 0; s < n_sc; ++s) {
        const vpmc_scenario sc = scs[s];
        if (!(sc.rsp_scale > 0)) FAIL(h, VPMC_ERR_INVALID_ARG, "scenario %d: rsp_scale must be positive", s);
        int rc = prepare_beams(h, sc, st); if (rc) return rc;
        const int ns = h->n_spots;
        const Ctx ctx = make_ctx(h, sc, seed);
        // S:8e: this handle's rows (vpmc_set_shard); the other rows stay empty
        const int g_lo = (int)((long long)ns * h->shard_index / h->shard_count), g_hi = (int)((long long)ns * (h->shard_index + 1) / h->shard_count);
        // ---- 1. pilot bounding boxes
        std::vector<int> bb((size_t)ns * 6);
        for (int g = 0; g < ns; ++g) { bb[6 * g] = bb[6 * g + 1] = bb[6 * g + 2] = 0x7fffffff; bb[6 * g + 3] = bb[6 * g + 4] = bb[6 * g + 5] = -1; }
        rc = upload(h, h->inf_bbox, bb, st); if (rc) return rc;
        {
            WorkMap wm{};
            wm.mode = 1; wm.hps = hist_per_spot; wm.n_sub = n_pilot; wm.cols = nullptr; wm.g0 = g_lo;
            wm.n_items = (unsigned long long)(g_hi - g_lo) * n_pilot;
            ScoreArgs sa{};
            sa.cb.bbox = h->inf_bbox.as<int>(); sa.sg = score_geom(h);
            CU(h, cudaMemsetAsync(h->d_tal_scratch, 0, sizeof(DevTallies), st));
            rc = launch_transport<2>(h, ctx, wm, sa, h->d_tal_scratch, st); if (rc) return rc;
        }
        CU(h, cudaMemcpyAsync(bb.data(), h->inf_bbox.p, bb.size() * sizeof(int), cudaMemcpyDeviceToHost, st));
        CU(h, cudaStreamSynchronize(st));
        // ---- 2. boxes
        std::vector<HostBox> box(ns);
        for (int g = g_lo; g < g_hi; ++g) {           // the pilot's columns are local: column c = spot g_lo + c
            const int *pb = &bb[6 * (size_t)(g - g_lo)];
            if (pb[3] < 0) { for (int a = 0; a < 3; ++a) { box[g].lo[a] = 0; box[g].dim[a] = 1; } }   // pilot deposited nothing
            else box[g] = grown_box(pb, h->sn, h->box_grow, h->box_pad);
        }
        // ---- 3./4. groups, with replay of the columns that outgrew their box
        std::vector<long long> row_nnz(ns, 0), row_src(ns, 0), row_ovf_off(ns, 0);
        std::vector<int> row_ovf_n(ns, 0);
        long long staged = 0, ostaged = 0;
        std::vector<int> todo(g_hi - g_lo);
        std::iota(todo.begin(), todo.end(), g_lo);
        bool replay = false;
        for (int round = 0; !todo.empty(); ++round) {
            if (round > 4) FAIL(h, VPMC_ERR_STATE, "influence: columns still outgrow their boxes after %d replays", round - 1);
            std::vector<int> next;
            size_t i0 = 0;
            while (i0 < todo.size()) {
                // pack a group
                std::vector<int> cols; std::vector<int4> lo, dim; std::vector<unsigned long long> off; std::vector<int> tile0(1, 0);
                long long elems = 0;
                while (i0 < todo.size()) {
                    const HostBox &b = box[todo[i0]];
                    const long long v8 = (b.vol() + 7) / 8 * 8;
                    if (!cols.empty() && (elems + v8 > limit_elems || cols.size() >= (1u << 24) - 1)) break;
                    cols.push_back(todo[i0]);
                    lo.push_back(make_int4(b.lo[0], b.lo[1], b.lo[2], 0)); dim.push_back(make_int4(b.dim[0], b.dim[1], b.dim[2], 0));
                    off.push_back((unsigned long long)elems);
                    tile0.push_back(tile0.back() + (int)((b.vol() + kTile - 1) / kTile));
                    elems += v8;
                    ++i0;
                }
                const int nc = (int)cols.size();
                h->inf_stats.box_elements += (uint64_t)elems; h->inf_stats.groups += 1;
                rc = ensure(h, h->inf_scratch, (size_t)elems * sizeof(float)); if (rc) return rc;
                std::vector<int> obb((size_t)nc * 6);
                for (int c = 0; c < nc; ++c) { obb[6 * c] = obb[6 * c + 1] = obb[6 * c + 2] = 0x7fffffff; obb[6 * c + 3] = obb[6 * c + 4] = obb[6 * c + 5] = -1; }
                if ((rc = upload(h, h->inf_cols, cols, st)) || (rc = upload(h, h->inf_lo, lo, st)) || (rc = upload(h, h->inf_dim, dim, st)) ||
                    (rc = upload(h, h->inf_off, off, st)) || (rc = upload(h, h->inf_tile0, tile0, st)) || (rc = upload(h, h->inf_bbox, obb, st))) return rc;
                CU(h, cudaMemsetAsync(h->inf_scratch.p, 0, (size_t)elems * sizeof(float), st));
                ColumnBoxes cb{};
                cb.lo = h->inf_lo.as<int4>(); cb.dim = h->inf_dim.as<int4>(); cb.offset = h->inf_off.as<unsigned long long>();
                cb.scratch = h->inf_scratch.as<float>(); cb.bbox = h->inf_bbox.as<int>();
                // overflow list: deposits outside the boxes (ovf_ctr[0]: entries appended)
                if ((rc = ensure(h, h->ovf_key, (size_t)ovf_cap * 8 + 8)) || (rc = ensure(h, h->ovf_val, (size_t)ovf_cap * 4 + 4)) ||
                    (rc = ensure(h, h->ovf_ctr, 4 * sizeof(int)))) return rc;
                CU(h, cudaMemsetAsync(h->ovf_ctr.p, 0, 4 * sizeof(int), st));
                cb.ovf_key = h->ovf_key.as<unsigned long long>(); cb.ovf_val = h->ovf_val.as<float>();
                cb.ovf_count = h->ovf_ctr.as<unsigned int>(); cb.ovf_cap = ovf_cap;
                {
                    WorkMap wm{};
                    wm.mode = 1; wm.hps = hist_per_spot; wm.n_sub = hist_per_spot; wm.cols = h->inf_cols.as<int>(); wm.g0 = 0;
                    wm.n_items = (unsigned long long)nc * hist_per_spot;
                    ScoreArgs sa{};
                    sa.cb = cb; sa.sg = score_geom(h);
                    if (replay) CU(h, cudaMemsetAsync(h->d_tal_scratch, 0, sizeof(DevTallies), st));
                    rc = launch_transport<1>(h, ctx, wm, sa, replay ? h->d_tal_scratch : h->d_tal, st); if (rc) return rc;
                }
                // which columns lost outside deposits (overflow list full): those are replayed with a larger box
                unsigned int n_ovf = 0;
                CU(h, cudaMemcpyAsync(obb.data(), h->inf_bbox.p, obb.size() * sizeof(int), cudaMemcpyDeviceToHost, st));
                CU(h, cudaMemcpyAsync(&n_ovf, h->ovf_ctr.p, sizeof(unsigned int), cudaMemcpyDeviceToHost, st));
                CU(h, cudaStreamSynchronize(st));
                n_ovf = std::min(n_ovf, ovf_cap);            // slots handed out, sentinels of the warps' unused stretches included
                // overflow entries per column; a column with more than a CTA sorts is treated like one that lost deposits
                std::vector<unsigned int> ovf_cnt(nc, 0u), ovf_off(nc, 0u);
                if (n_ovf > 0) {
                    if ((rc = ensure(h, h->ovf_colcnt, (size_t)nc * 4)) || (rc = ensure(h, h->ovf_flag, (size_t)nc * 4)) || (rc = ensure(h, h->ovf_kept, (size_t)nc * 4))) return rc;
                    const int g1 = std::max(1, std::min((int)((n_ovf + 255) / 256), h->n_sm * 8));
                    CU(h, cudaMemsetAsync(h->ovf_colcnt.p, 0, (size_t)nc * 4, st));
                    ovf_hist_kernel<<<g1, 256, 0, st>>>(h->ovf_key.as<unsigned long long>(), n_ovf, h->ovf_colcnt.as<unsigned int>());
                    h->launches += 1;
                    CU(h, cudaMemcpyAsync(ovf_cnt.data(), h->ovf_colcnt.p, (size_t)nc * 4, cudaMemcpyDeviceToHost, st));
                    CU(h, cudaStreamSynchronize(st));
                    std::vector<int> big(nc, 0);
                    bool any_big = false;
                    unsigned int run = 0;
                    for (int c = 0; c < nc; ++c) { ovf_off[c] = run; run += ovf_cnt[c]; if (ovf_cnt[c] > h->ovf_sort_cap) { big[c] = 1; any_big = true; } }
                    h->inf_stats.ovf_deposits += run;
                    if (any_big) {
                        rc = upload(h, h->inf_skip, big, st); if (rc) return rc;
                        ovf_bbox_kernel<<<g1, 256, 0, st>>>(h->ovf_key.as<unsigned long long>(), n_ovf, h->inf_skip.as<int>(), h->sn[0], h->sn[1], h->inf_bbox.as<int>());
                        h->launches += 1;
                        CU(h, cudaMemcpyAsync(obb.data(), h->inf_bbox.p, obb.size() * sizeof(int), cudaMemcpyDeviceToHost, st));
                        CU(h, cudaStreamSynchronize(st));
                    }
                }
                std::vector<int> skip(nc, 0);
                for (int c = 0; c < nc; ++c)
                    if (obb[6 * c + 3] >= 0) {
                        skip[c] = 1;
                        HostBox &b = box[cols[c]];
                        int u[6];
                        for (int a = 0; a < 3; ++a) { u[a] = std::min(b.lo[a], obb[6 * c + a]); u[3 + a] = std::max(b.lo[a] + b.dim[a] - 1, obb[6 * c + 3 + a]); }
                        for (int a = 0; a < 3; ++a) { b.lo[a] = u[a]; b.dim[a] = u[3 + a] - u[a] + 1; }
                        next.push_back(cols[c]);
                        h->inf_stats.columns_replayed += 1;
                    }
                rc = upload(h, h->inf_skip, skip, st); if (rc) return rc;
                CsrCols cc{};
                cc.lo = cb.lo; cc.dim = cb.dim; cc.offset = cb.offset; cc.tile0 = h->inf_tile0.as<int>(); cc.skip = h->inf_skip.as<int>();
                cc.n_cols = nc; cc.n_tiles = tile0.back(); cc.nx = h->sn[0]; cc.ny = h->sn[1];
                cc.tile_col = nullptr;
                if (cc.n_tiles > 0) {
                    rc = ensure(h, h->inf_tilecol, (size_t)cc.n_tiles * sizeof(int)); if (rc) return rc;
                    csr_tile_cols_kernel<<<(cc.n_tiles + 255) / 256, 256, 0, st>>>(cc, h->inf_tilecol.as<int>());
                    cc.tile_col = h->inf_tilecol.as<int>();
                    h->launches += 1;
                }
                rc = csr_max_pass(h, cc, cb.scratch, true, coef, st); if (rc) return rc;
                std::vector<unsigned int> ocnt(nc, 0u);
                if (n_ovf > 0) {
                    // bucket by column, then one CTA per column: sort by cell, sum per cell, convert, column maximum, threshold,
                    // kept pairs written at the start of the column's stretch of the overflow staging (vpmc_kernels.cuh)
                    if ((rc = ensure(h, h->ovf_key2, (size_t)n_ovf * 4)) || (rc = ensure(h, h->ovf_val2, (size_t)n_ovf * 4)) ||
                        (rc = grow_keep(h, h->ostage_idx, (size_t)(ostaged + n_ovf) * sizeof(int), (size_t)ostaged * sizeof(int), st)) ||
                        (rc = grow_keep(h, h->ostage_val, (size_t)(ostaged + n_ovf) * sizeof(float), (size_t)ostaged * sizeof(float), st)) ||
                        (rc = upload(h, h->ovf_coloff, ovf_off, st))) return rc;
                    static bool smem_set = false;
                    if (!smem_set) { CU(h, cudaFuncSetAttribute(ovf_columns_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kOvfSortCap * 8)); smem_set = true; }
                    TimedScope ts(h, st, 3);
                    const int g1 = std::max(1, std::min((int)((n_ovf + 255) / 256), h->n_sm * 8));
                    CU(h, cudaMemsetAsync(h->ovf_flag.p, 0, (size_t)nc * 4, st));                // cursors
                    ovf_scatter_kernel<<<g1, 256, 0, st>>>(h->ovf_key.as<unsigned long long>(), h->ovf_val.as<float>(), n_ovf, h->ovf_coloff.as<unsigned int>(),
                                                          h->ovf_flag.as<unsigned int>(), h->ovf_key2.as<unsigned int>(), h->ovf_val2.as<float>());
                    ovf_columns_kernel<<<nc, kOvfBlock, kOvfSortCap * 8, st>>>(h->ovf_key2.as<unsigned int>(), h->ovf_val2.as<float>(), h->ovf_coloff.as<unsigned int>(),
                                                                           h->ovf_colcnt.as<unsigned int>(), h->inf_skip.as<int>(), h->d_hu, h->d_lut, h->G.hu_min, h->G.n_lut,
                                                                           h->params.rho_min, coef, h->d_cell_rho, rel_threshold, h->inf_colmax.as<unsigned int>(),
                                                                           h->ostage_idx.as<int>() + ostaged, h->ostage_val.as<float>() + ostaged, h->ovf_kept.as<unsigned int>(), h->ovf_sort_cap);
                    CU(h, cudaGetLastError());
                    h->launches += 2;
                    CU(h, cudaMemcpyAsync(ocnt.data(), h->ovf_kept.p, (size_t)nc * 4, cudaMemcpyDeviceToHost, st));
                }
                rc = csr_count_pass(h, cc, cb.scratch, rel_threshold, st); if (rc) return rc;
                std::vector<long long> nnz(nc), base(nc);
                CU(h, cudaMemcpyAsync(nnz.data(), h->inf_colnnz.p, (size_t)nc * sizeof(long long), cudaMemcpyDeviceToHost, st));
                CU(h, cudaStreamSynchronize(st));
                long long add = 0, oadd = 0;
                for (int c = 0; c < nc; ++c) {
                    base[c] = staged + add;
                    if (!skip[c]) {
                        row_nnz[cols[c]] = nnz[c] + ocnt[c]; row_src[cols[c]] = base[c]; add += nnz[c];
                        row_ovf_off[cols[c]] = ostaged + (long long)(n_ovf > 0 ? ovf_off[c] : 0u); row_ovf_n[cols[c]] = (int)ocnt[c]; oadd += ocnt[c];
                    }
                }
                if (n_ovf > 0) ostaged += n_ovf;          // a column's kept pairs sit at the start of its bucket's stretch
                h->inf_stats.ovf_kept += (uint64_t)oadd;
                if (h->verbose) fprintf(stderr, "[vpmc]   group of %d columns: %u outside deposits, %lld kept entries of them, %lld box entries\n", nc, n_ovf, oadd, add);
                if (add > 0) {
                    if ((rc = grow_keep(h, h->inf_stage_idx, (size_t)(staged + add) * sizeof(int), (size_t)staged * sizeof(int), st)) ||
                        (rc = grow_keep(h, h->inf_stage_val, (size_t)(staged + add) * sizeof(float), (size_t)staged * sizeof(float), st)) ||
                        (rc = upload(h, h->inf_colbase, base, st))) return rc;
                    TimedScope ts(h, st, 3);
                    csr_emit_kernel<<<tile_grid(h, (const void *)csr_emit_kernel, cc.n_tiles), kBlock, 0, st>>>(cc, cb.scratch, h->inf_colmax.as<unsigned int>(), rel_threshold,
                                                                                                     h->inf_tilecnt.as<unsigned int>(), h->inf_colbase.as<long long>(),
                                                                                                     h->inf_stage_idx.as<int>(), h->inf_stage_val.as<float>());
                    CU(h, cudaGetLastError());
                    h->launches += 1;
                    staged += add;
                }
            }
            if (h->verbose) fprintf(stderr, "[vpmc] influence scenario %d round %d: %zu columns, %zu to replay\n", s, round, todo.size(), next.size());
            todo.swap(next);
            replay = true;
        }
        // ---- 5. assemble this scenario's CSR in caller-owned memory
        std::vector<long long> row_ptr(ns + 1, 0);
        for (int g = 0; g < ns; ++g) row_ptr[g + 1] = row_ptr[g] + row_nnz[g];
        const long long nnz = row_ptr[ns];
        vpmc_csr &o = out[s];
        o.n_rows = ns; o.nnz = nnz;
        h->inf_stats.nnz += (uint64_t)nnz;
        o.row_ptr = (int64_t *)alloc((size_t)(ns + 1) * sizeof(int64_t), user);
        o.col = (int32_t *)alloc((size_t)std::max<long long>(nnz, 1) * sizeof(int32_t), user);
        o.val = (float *)alloc((size_t)std::max<long long>(nnz, 1) * sizeof(float), user);
        if (!o.row_ptr || !o.col || !o.val) FAIL(h, VPMC_ERR_ALLOC, "the caller's allocator returned NULL (scenario %d, nnz %lld)", s, nnz);
        CU(h, cudaMemcpyAsync(o.row_ptr, row_ptr.data(), (size_t)(ns + 1) * sizeof(int64_t), cudaMemcpyHostToDevice, st));
        if ((rc = upload(h, h->inf_rowsrc, row_src, st)) || (rc = upload(h, h->row_ovf_off, row_ovf_off, st)) || (rc = upload(h, h->row_ovf_n, row_ovf_n, st))) return rc;
        if (nnz > 0) {
            TimedScope ts(h, st, 3);
            csr_gather_rows_kernel<<<std::min(ns, h->n_sm * 8), 256, 0, st>>>(ns, h->inf_rowsrc.as<long long>(), h->row_ovf_off.as<long long>(), h->row_ovf_n.as<int>(),
                                                                             (const long long *)o.row_ptr, h->inf_stage_idx.as<int>(), h->inf_stage_val.as<float>(),
                                                                             h->ostage_idx.as<int>(), h->ostage_val.as<float>(), o.col, o.val);
            CU(h, cudaGetLastError());
            h->launches += 1;
        }
        CU(h, cudaStreamSynchronize(st));     // row_ptr / row_src host vectors go out of scope; outputs are final
    }
    return VPMC_OK;
}
