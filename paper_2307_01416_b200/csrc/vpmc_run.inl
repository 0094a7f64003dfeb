// vpmc_run.inl -- launch sequencing of the dose path (included by vpmc_api.cu).

// C2: largest-remainder apportionment of N histories to the spot weights (integer-exact)
static void apportion(unsigned long long N, const std::vector<double> &w, std::vector<unsigned long long> &cnt)
{
    const size_t n = w.size();
    cnt.assign(n, 0ull);
    double W = 0.0;
    for (double x : w) W += x;
    std::vector<double> frac(n, 0.0);
    unsigned long long assigned = 0;
    for (size_t j = 0; j < n; ++j) {
        const double q = (W > 0.0) ? (double)N * w[j] / W : 0.0;
        const double f = std::floor(q);
        cnt[j] = (unsigned long long)f;
        frac[j] = q - f;
        assigned += cnt[j];
    }
    unsigned long long left = N > assigned ? N - assigned : 0;
    if (n == 0) return;
    std::vector<size_t> order(n);
    std::iota(order.begin(), order.end(), (size_t)0);
    std::stable_sort(order.begin(), order.end(), [&](size_t a, size_t b) { return frac[a] > frac[b]; });
    for (size_t k = 0; left > 0; k = (k + 1) % n, --left) cnt[order[k]] += 1;
}

// most upstream w of the (shifted) CT box corners in the beam frame
static double ct_min_w(const vpmc_t *h, const BeamHost &b, const float shift[3])
{
    const DevGrid &G = h->G;
    const double lo[3] = { G.ox, G.oy, G.oz };
    const double hi[3] = { (double)G.ox + (double)G.nx * G.hx, (double)G.oy + (double)G.ny * G.hy, (double)G.oz + (double)G.nz * G.hz };
    double wmin = std::numeric_limits<double>::infinity();
    for (int k = 0; k < 8; ++k) {
        double c[3];
        for (int a = 0; a < 3; ++a) c[a] = (((k >> a) & 1) ? hi[a] : lo[a]) - ((double)b.frame.iso[a] - (double)shift[a]);
        const double w = (double)b.frame.rot[2] * c[0] + (double)b.frame.rot[5] * c[1] + (double)b.frame.rot[8] * c[2];
        wmin = std::min(wmin, w);
    }
    return wmin;
}

// upload spots (once per change) and the per-scenario beam descriptors
static int prepare_beams(vpmc_t *h, const vpmc_scenario &sc, cudaStream_t st)
{
    if (h->beams.empty()) FAIL(h, VPMC_ERR_STATE, "no beam");
    join_setup(h, st);
    h->launched = true;
    if (h->spots_dirty) {
        std::vector<float4> sp;
        std::vector<double> r0;
        h->spot_w.clear(); h->spot_beam_h.clear();
        for (size_t b = 0; b < h->beams.size(); ++b)
            for (const vpmc_spot &s : h->beams[b].spots) {
                sp.push_back(make_float4(s.x, s.y, s.energy, s.sigma));
                r0.push_back((double)h->params.alpha * std::pow((double)s.energy, (double)h->params.p));   // S0: R0 = alpha E^p in fp64
                h->spot_w.push_back((double)s.weight);
                h->spot_beam_h.push_back((int)b);
            }
        h->n_spots = (int)sp.size();
        if (h->n_spots == 0) FAIL(h, VPMC_ERR_STATE, "no spots");
        dev_release(h, h->d_spots); dev_release(h, h->d_spot_R0); dev_release(h, h->d_spot_beam); dev_release(h, h->d_beams);
        h->d_spots = nullptr; h->d_spot_R0 = nullptr; h->d_spot_beam = nullptr; h->d_beams = nullptr;
        int rc;
        if ((rc = dev_alloc(h, (void **)&h->d_spots, sp.size() * sizeof(float4))) || (rc = dev_alloc(h, (void **)&h->d_spot_R0, r0.size() * sizeof(double))) ||
            (rc = dev_alloc(h, (void **)&h->d_spot_beam, sp.size() * sizeof(int))) || (rc = dev_alloc(h, (void **)&h->d_beams, h->beams.size() * sizeof(DevBeam)))) return rc;
        CU(h, cudaMemcpyAsync(h->d_spots, sp.data(), sp.size() * sizeof(float4), cudaMemcpyHostToDevice, st));
        CU(h, cudaMemcpyAsync(h->d_spot_R0, r0.data(), r0.size() * sizeof(double), cudaMemcpyHostToDevice, st));
        CU(h, cudaMemcpyAsync(h->d_spot_beam, h->spot_beam_h.data(), sp.size() * sizeof(int), cudaMemcpyHostToDevice, st));
        h->spots_dirty = false;
    }
    std::vector<DevBeam> db(h->beams.size());
    for (size_t i = 0; i < h->beams.size(); ++i) {
        const BeamHost &b = h->beams[i];
        DevBeam &d = db[i];
        memset(&d, 0, sizeof(d));
        memcpy(d.iso, b.frame.iso, sizeof(d.iso));
        memcpy(d.rot, b.frame.rot, sizeof(d.rot));
        d.has_rs = b.rs_wet > 0.0f;
        d.w_rs_out = -b.rs_face;
        d.w_rs_in = d.w_rs_out - b.rs_wet / h->params.rs_rsp;
        d.has_ap = b.has_ap;
        d.w_ap_out = -b.ap_face;
        d.w_ap_in = d.w_ap_out - b.ap_T;
        d.ap_bits = b.d_bits; d.ap_nx = b.ap_nx; d.ap_ny = b.ap_ny; d.ap_row_words = b.ap_row_words;
        d.ap_u0 = b.ap_u0; d.ap_v0 = b.ap_v0; d.ap_inv_du = (float)(1.0 / (double)b.ap_du); d.ap_inv_dv = (float)(1.0 / (double)b.ap_dv);
        d.ap_dist = b.d_dist; d.ap_dist_open = b.d_dist ? b.d_dist + (size_t)b.ap_ntx * b.ap_nty : nullptr; d.ap_ntx = b.ap_ntx;
        d.ap_tile_u = (float)(1 << kApTileShift) * b.ap_du; d.ap_tile_v = (float)(1 << kApTileShift) * b.ap_dv;
        d.ap_poly = b.d_poly; d.ap_n_poly = b.ap_n_poly; d.ap_pgrid = b.d_pgrid; d.ap_pg_nx = b.pg_nx; d.ap_pg_ny = b.pg_ny;
        d.ap_pg_x0 = b.pg_x0; d.ap_pg_y0 = b.pg_y0; d.ap_pg_inv_cell = (float)(1.0 / (double)b.pg_cell);
        d.ap_prow_ptr = b.d_prows; d.ap_pedges = b.d_prows ? b.d_prows + b.pg_ny + 1 : nullptr;
        const double wct = ct_min_w(h, b, sc.shift);
        if (d.has_rs && d.has_ap && d.w_rs_out > d.w_ap_in) FAIL(h, VPMC_ERR_GEOMETRY, "beam %zu: range shifter is not upstream of the aperture", i);
        const double w_last = d.has_ap ? d.w_ap_out : (d.has_rs ? d.w_rs_out : -std::numeric_limits<double>::infinity());
        if (wct < w_last) FAIL(h, VPMC_ERR_GEOMETRY, "beam %zu: the CT box overlaps the beam-line devices", i);
        if (d.has_rs) d.w_start = d.w_rs_in - 1.0f;
        else if (d.has_ap) d.w_start = d.w_ap_in - 1.0f;
        else d.w_start = (float)(wct - 1.0);
    }
    CU(h, cudaMemcpyAsync(h->d_beams, db.data(), db.size() * sizeof(DevBeam), cudaMemcpyHostToDevice, st));
    return VPMC_OK;
}

static Ctx make_ctx(const vpmc_t *h, const vpmc_scenario &sc, uint64_t seed)
{
    Ctx c;
    c.P = h->P; c.G = h->G; c.beams = h->d_beams; c.hu = h->d_hu;
    c.rsp_scale = sc.rsp_scale; c.inv_rsp_scale = (float)(1.0 / (double)sc.rsp_scale);
    c.shift[0] = sc.shift[0]; c.shift[1] = sc.shift[1]; c.shift[2] = sc.shift[2];
    for (int r = 0; r < 10; ++r) { c.K.k0[r] = (uint32_t)seed + (uint32_t)r * 0x9E3779B9u; c.K.k1[r] = (uint32_t)(seed >> 32) + (uint32_t)r * 0xBB67AE85u; }
    return c;
}

// buffers of one chunk of `cap` work items: range-shifter records, the three queues
struct ChunkBufs { SourceBuf sb; Queue q_rs_out, q_ap, q_ct; unsigned int *rs_head, *ap_head; };

static int chunk_buffers(vpmc_t *h, unsigned long long cap, ChunkBufs &cb)
{
    bool any_rs = false, any_ap = false;
    for (const BeamHost &b : h->beams) { any_rs = any_rs || b.rs_wet > 0.0f; any_ap = any_ap || b.has_ap; }
    h->any_rs = any_rs; h->any_ap = any_ap;
    int rc;
    DevBuf *ct[5] = { &h->q0, &h->q1, &h->q2, &h->q3, &h->q4 };
    for (DevBuf *b : ct) if ((rc = ensure(h, *b, cap * 16))) return rc;
    if (any_rs) {
        DevBuf *rs[8] = { &h->s0, &h->s1, &h->s2, &h->a0, &h->a1, &h->a2, &h->a3, &h->a4 };
        for (DevBuf *b : rs) if ((rc = ensure(h, *b, cap * 16))) return rc;
    }
    if (any_ap) {
        DevBuf *ap[6] = { &h->b0, &h->b1, &h->b2, &h->b3, &h->b4, &h->b5 };
        for (DevBuf *b : ap) if ((rc = ensure(h, *b, cap * 16))) return rc;
    }
    unsigned int *ctr = h->d_qctr;      // [0] CT count, [1] CT head, [2] rs records, [3] rs head, [4] rs-out count, [5] ap count, [6] ap head
    cb.sb.s0 = h->s0.as<uint4>(); cb.sb.s1 = h->s1.as<uint4>(); cb.sb.s2 = h->s2.as<uint4>(); cb.sb.count = ctr + 2;
    cb.rs_head = ctr + 3; cb.ap_head = ctr + 6;
    Queue &z = cb.q_ct;
    z.q0 = h->q0.as<uint4>(); z.q1 = h->q1.as<float4>(); z.q2 = h->q2.as<float4>(); z.q3 = h->q3.as<uint4>(); z.q4 = h->q4.as<uint4>(); z.q5 = nullptr;
    z.count = ctr; z.head = ctr + 1; z.capacity = (unsigned int)cap;
    Queue &a = cb.q_rs_out;
    a.q0 = h->a0.as<uint4>(); a.q1 = h->a1.as<float4>(); a.q2 = h->a2.as<float4>(); a.q3 = h->a3.as<uint4>(); a.q4 = h->a4.as<uint4>(); a.q5 = nullptr;
    a.count = ctr + 4; a.head = nullptr; a.capacity = (unsigned int)cap;
    Queue &b = cb.q_ap;
    b.q0 = h->b0.as<uint4>(); b.q1 = h->b1.as<float4>(); b.q2 = h->b2.as<float4>(); b.q3 = h->b3.as<uint4>(); b.q4 = h->b4.as<uint4>(); b.q5 = h->b5.as<float4>();
    b.count = ctr + 5; b.head = ctr + 6; b.capacity = (unsigned int)cap;
    return VPMC_OK;
}

// one chunk of the hot path on stream st: source + opening phase (S1, S3) -> range shifter (S2) -> aperture entry -> brass
// (S3) -> CT entry -> voxel stepping + scoring (S4-S7).  Plain launches, so the sequence can also be captured into a graph.
template <int MODE>
static void enqueue_chunk(vpmc_t *h, const Ctx &c, const WorkMap &wm, unsigned long long i0, const ChunkBufs &cb, const ScoreArgs &sa,
                          DevTallies *tal, cudaStream_t st, bool timed)
{
    const unsigned int n = (unsigned int)wm.n_items;
    const int blocks = (int)((n + kBlock - 1) / kBlock);
    cudaMemsetAsync(h->d_qctr, 0, 8 * sizeof(unsigned int), st);
    // timing classes: 4 = the one-thread-per-item stage kernels, 0 = the persistent beam-line kernels, 1 = the voxel kernel
    {
        TimedScope ts(h, st, 4, timed);
        source_kernel<<<blocks, kBlock, 0, st>>>(c, wm, i0, h->d_spots, h->d_spot_R0, h->d_spot_beam, cb.sb, cb.q_ap, cb.q_ct, tal);
    }
    if (h->any_rs) {
        {
            TimedScope ts(h, st, 0, timed);
            beam_fn(0, h->fl)<<<std::min(h->grid_beam[0][h->fl], blocks), kBlock, 0, st>>>(c, cb.sb, cb.q_rs_out, cb.q_rs_out, cb.rs_head, tal);
        }
        TimedScope ts(h, st, 4, timed);
        ap_entry_kernel<<<blocks, kBlock, 0, st>>>(c, cb.q_rs_out, cb.q_ap, cb.q_ct, tal);
    }
    if (h->any_ap) {
        TimedScope ts(h, st, 0, timed);
        beam_fn(1, h->fl)<<<std::min(h->grid_beam[1][h->fl], blocks), kBlock, 0, st>>>(c, cb.sb, cb.q_ap, cb.q_ct, cb.ap_head, tal);
    }
    {
        TimedScope ts(h, st, 4, timed);
        entry_kernel<<<blocks, kBlock, 0, st>>>(c, cb.q_ct, tal);
    }
    TimedScope ts(h, st, 1, timed);
    const int sl = h->smem_lut ? 1 : 0;
    voxel_fn(MODE, sl, h->fl)<<<std::min(h->grid[MODE][sl][h->fl], blocks), kBlock, h->tally_smem + (sl ? h->lut_bytes : 0), st>>>(c, cb.q_ct, h->d_lut, sa, tal);
}

static unsigned int chunk_launches(const vpmc_t *h) { return 3u + (h->any_rs ? 2u : 0u) + (h->any_ap ? 1u : 0u); }

// the hot path over wm.n_items work items, in chunks of h->chunk
template <int MODE>
static int launch_transport(vpmc_t *h, const Ctx &c, const WorkMap &wm0, const ScoreArgs &sa, DevTallies *tal, cudaStream_t st)
{
    if (wm0.n_items == 0) return VPMC_OK;
    const unsigned long long cap = std::min<unsigned long long>(wm0.n_items, h->chunk);
    ChunkBufs cb;
    int rc = chunk_buffers(h, cap, cb); if (rc) return rc;
    for (unsigned long long i0 = 0; i0 < wm0.n_items; i0 += h->chunk) {
        WorkMap wm = wm0;
        wm.n_items = std::min<unsigned long long>(h->chunk, wm0.n_items - i0);
        enqueue_chunk<MODE>(h, c, wm, i0, cb, sa, tal, st, true);
        CU(h, cudaGetLastError());
        h->launches += chunk_launches(h);
    }
    return VPMC_OK;
}

static int grid_for(long long n, int n_sm) { return (int)std::max<long long>(1, std::min<long long>((n + 255) / 256, (long long)n_sm * 16)); }

extern "C" int vpmc_dose_scenario(vpmc_t *h, const vpmc_scenario *scp, uint64_t n_histories, uint64_t seed,
                                  float *dose_out_dev, void *cuda_stream)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    if (!dose_out_dev || !scp) FAIL(h, VPMC_ERR_INVALID_ARG, "NULL argument");
    if (!(scp->rsp_scale > 0)) FAIL(h, VPMC_ERR_INVALID_ARG, "rsp_scale must be positive");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const vpmc_scenario sc = *scp;
    int rc = prepare_beams(h, sc, st); if (rc) return rc;
    h->last_stream = st;
    h->unc_valid = false;
    const int B = h->params.n_batches;
    const bool with_unc = B >= 2;
    if (with_unc && !h->d_s1) {
        if ((rc = dev_alloc(h, (void **)&h->d_s1, h->ncell * sizeof(float))) || (rc = dev_alloc(h, (void **)&h->d_s2, h->ncell * sizeof(float)))) return rc;
    }
    rc = ensure(h, h->edep, (size_t)B * h->ncell * sizeof(float)); if (rc) return rc;
    const size_t n_ent = (size_t)B * h->n_spots;
    rc = ensure(h, h->cum, (n_ent + 1) * sizeof(unsigned long long)); if (rc) return rc;
    rc = ensure(h, h->first, (n_ent + 1) * sizeof(unsigned long long)); if (rc) return rc;
    // C2: history ids are contiguous per spot in spot order; batch b takes sub-range b of every spot (R7)
    std::vector<unsigned long long> cnt, start(h->n_spots + 1, 0ull);
    apportion(n_histories, h->spot_w, cnt);
    for (int g = 0; g < h->n_spots; ++g) start[g + 1] = start[g] + cnt[g];
    const unsigned long long wlo = h->win_lo, whi = h->win_hi ? std::min<unsigned long long>(h->win_hi, n_histories) : n_histories;
    std::vector<unsigned long long> cum(n_ent + 1, 0ull), first(n_ent + 1, 0ull);
    std::vector<float> fb(B, 0.0f);
    std::vector<unsigned long long> nb(B, 0ull);
    for (int b = 0; b < B; ++b)
        for (int g = 0; g < h->n_spots; ++g) {
            const unsigned __int128 n = cnt[g];
            unsigned long long lo = start[g] + (unsigned long long)((n * (unsigned)b) / (unsigned)B);
            unsigned long long hi = start[g] + (unsigned long long)((n * (unsigned)(b + 1)) / (unsigned)B);
            if (h->shard_count > 1) {           // S:8e: shard k of K of every (spot, batch) id range
                const unsigned __int128 len = hi - lo;
                const unsigned long long a = lo + (unsigned long long)((len * (unsigned)h->shard_index) / (unsigned)h->shard_count);
                hi = lo + (unsigned long long)((len * (unsigned)(h->shard_index + 1)) / (unsigned)h->shard_count);
                lo = a;
            }
            lo = std::max(lo, wlo); hi = std::min(hi, whi);
            const size_t e = (size_t)b * h->n_spots + g;
            first[e] = lo;
            const unsigned long long k = hi > lo ? hi - lo : 0ull;
            cum[e + 1] = cum[e] + k;
            nb[b] += k;
        }
    const unsigned long long n_total = cum[n_ent];
    for (int b = 0; b < B; ++b) fb[b] = nb[b] ? (float)((double)n_total / (double)nb[b]) : 0.0f;

    CU(h, cudaMemsetAsync(h->edep.p, 0, (size_t)B * h->ncell * sizeof(float), st));
    CU(h, cudaMemsetAsync(h->d_tal, 0, sizeof(DevTallies), st));
    CU(h, cudaMemsetAsync(h->d_max_bits, 0, sizeof(unsigned int), st));
    CU(h, cudaMemsetAsync(h->d_unc, 0, 2 * sizeof(double), st));
    CU(h, cudaMemcpyAsync(h->cum.p, cum.data(), (n_ent + 1) * sizeof(unsigned long long), cudaMemcpyHostToDevice, st));
    CU(h, cudaMemcpyAsync(h->first.p, first.data(), (n_ent + 1) * sizeof(unsigned long long), cudaMemcpyHostToDevice, st));
    CU(h, cudaMemcpyAsync(h->d_fb, fb.data(), B * sizeof(float), cudaMemcpyHostToDevice, st));

    WorkMap wm{};
    wm.mode = 0; wm.n_items = n_total; wm.cum = h->cum.as<unsigned long long>(); wm.first = h->first.as<unsigned long long>();
    wm.n_entries = (int)n_ent; wm.n_spots = h->n_spots;
    ScoreArgs sa{};
    sa.edep = h->edep.as<float>(); sa.nvox = (unsigned long long)h->ncell; sa.sg = score_geom(h);
    rc = launch_transport<0>(h, make_ctx(h, sc, seed), wm, sa, h->d_tal, st); if (rc) return rc;
    // C6
    double W = 0.0;
    for (double x : h->spot_w) W += x;
    const double V = (double)h->G.hx * h->G.hy * h->G.hz * 1e-3;
    const float coef = (float)((n_histories ? W / (double)n_histories : 0.0) / V * 1.602176634e-10);
    TimedScope ts(h, st, 2);
    dose_finalize_kernel<<<grid_for(h->ncell, h->n_sm), 256, 0, st>>>(h->edep.as<float>(), B, h->d_fb, h->d_hu, h->d_lut, h->G, h->params.rho_min, coef,
                                                                   dose_out_dev, with_unc ? h->d_s1 : nullptr, with_unc ? h->d_s2 : nullptr, h->ncell, h->d_max_bits, h->d_cell_rho);
    CU(h, cudaGetLastError());
    h->launches += 1;
    if (with_unc) {
        uncertainty_kernel<<<grid_for(h->ncell, h->n_sm), 256, 0, st>>>(dose_out_dev, h->d_s1, h->d_s2, h->ncell, B, h->d_max_bits, h->d_unc);
        CU(h, cudaGetLastError());
        h->launches += 1;
        h->unc_valid = true;
    }
    return VPMC_OK;
}

extern "C" int vpmc_dose(vpmc_t *h, uint64_t n_histories, uint64_t seed, float *dose_out_dev, void *cuda_stream)
{
    const vpmc_scenario sc = { { 0.0f, 0.0f, 0.0f }, 1.0f };
    return vpmc_dose_scenario(h, &sc, n_histories, seed, dose_out_dev, cuda_stream);
}

extern "C" int vpmc_dose_host(vpmc_t *h, uint64_t n_histories, uint64_t seed, float *dose_out_host)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    if (!dose_out_host) FAIL(h, VPMC_ERR_INVALID_ARG, "NULL argument");
    DevBuf tmp;
    int rc = ensure(h, tmp, h->ncell * sizeof(float)); if (rc) return rc;
    float *d = tmp.as<float>();
    rc = vpmc_dose(h, n_histories, seed, d, nullptr);
    if (rc == VPMC_OK) {
        cudaError_t e = cudaMemcpy(dose_out_host, d, h->ncell * sizeof(float), cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) { h->err = cudaGetErrorString(e); rc = VPMC_ERR_CUDA; }
    }
    pool_give(tmp.p, tmp.bytes);
    return rc;
}

// ---- S:8f-3: dose to a statistical uncertainty, stopping rule on the device (CUDA-graph WHILE node)
static void seq_release(vpmc_t *h)
{
    if (h->seq_exec) { cudaGraphExecDestroy(h->seq_exec); h->seq_exec = nullptr; }
    if (h->seq_graph) { cudaGraphDestroy(h->seq_graph); h->seq_graph = nullptr; }
}

extern "C" int vpmc_dose_to_uncertainty(vpmc_t *h, const vpmc_scenario *scp, uint64_t batch_histories, int32_t min_batches,
                                        int32_t max_batches, float target_rel_unc, uint64_t seed, float *dose_out_dev, void *cuda_stream)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    if (!dose_out_dev || batch_histories < 1 || batch_histories > h->chunk || batch_histories >= (1ull << 32) || max_batches < 1 ||
        min_batches < 0 || !(target_rel_unc >= 0.0f))
        FAIL(h, VPMC_ERR_INVALID_ARG, "bad dose_to_uncertainty arguments (batch_histories must be in [1, chunk = %llu])", h->chunk);
    const vpmc_scenario sc = scp ? *scp : vpmc_scenario{ { 0, 0, 0 }, 1.0f };
    if (!(sc.rsp_scale > 0)) FAIL(h, VPMC_ERR_INVALID_ARG, "rsp_scale must be positive");
    cudaStream_t caller = (cudaStream_t)cuda_stream;
    if (!h->seq_stream) {
        CU(h, cudaStreamCreateWithFlags(&h->seq_stream, cudaStreamNonBlocking));
        CU(h, cudaEventCreateWithFlags(&h->seq_ev_in, cudaEventDisableTiming));
        CU(h, cudaEventCreateWithFlags(&h->seq_ev_out, cudaEventDisableTiming));
        int rc0 = dev_alloc(h, (void **)&h->d_seq, sizeof(SeqState)); if (rc0) return rc0;
    }
    cudaStream_t st = h->seq_stream;
    CU(h, cudaStreamSynchronize(st));        // a previous graph of this handle must have drained before it is rebuilt
    seq_release(h);
    CU(h, cudaEventRecord(h->seq_ev_in, caller));
    CU(h, cudaStreamWaitEvent(st, h->seq_ev_in, 0));
    int rc = prepare_beams(h, sc, st); if (rc) return rc;
    h->last_stream = caller;
    h->unc_valid = false; h->seq_valid = false;
    if (!h->d_s1) {
        if ((rc = dev_alloc(h, (void **)&h->d_s1, h->ncell * sizeof(float))) || (rc = dev_alloc(h, (void **)&h->d_s2, h->ncell * sizeof(float)))) return rc;
    }
    ChunkBufs cb;
    if ((rc = ensure(h, h->edep, (size_t)h->ncell * sizeof(float))) ||
        (rc = ensure(h, h->cum, ((size_t)h->n_spots + 1) * sizeof(unsigned long long))) || (rc = ensure(h, h->first, ((size_t)h->n_spots + 1) * sizeof(unsigned long long))) ||
        (rc = chunk_buffers(h, batch_histories, cb))) return rc;
    // C2 for one batch: ids i in [0, N_b) contiguous per spot in spot order (the batch index goes into the id's high word)
    std::vector<unsigned long long> cnt, cum(h->n_spots + 1, 0ull), first(h->n_spots + 1, 0ull);
    apportion(batch_histories, h->spot_w, cnt);
    for (int g = 0; g < h->n_spots; ++g) { first[g] = cum[g]; cum[g + 1] = cum[g] + cnt[g]; }
    CU(h, cudaMemcpyAsync(h->cum.p, cum.data(), cum.size() * sizeof(unsigned long long), cudaMemcpyHostToDevice, st));
    CU(h, cudaMemcpyAsync(h->first.p, first.data(), first.size() * sizeof(unsigned long long), cudaMemcpyHostToDevice, st));
    CU(h, cudaStreamSynchronize(st));        // cum / first are stack vectors
    CU(h, cudaMemsetAsync(h->edep.p, 0, (size_t)h->ncell * sizeof(float), st));
    CU(h, cudaMemsetAsync(h->d_s1, 0, (size_t)h->ncell * sizeof(float), st));
    CU(h, cudaMemsetAsync(h->d_s2, 0, (size_t)h->ncell * sizeof(float), st));
    CU(h, cudaMemsetAsync(h->d_tal, 0, sizeof(DevTallies), st));
    CU(h, cudaMemsetAsync(h->d_seq, 0, sizeof(SeqState), st));

    const Ctx c = make_ctx(h, sc, seed);
    WorkMap wm{};
    wm.mode = 0; wm.n_items = batch_histories; wm.cum = h->cum.as<unsigned long long>(); wm.first = h->first.as<unsigned long long>();
    wm.n_entries = h->n_spots; wm.n_spots = h->n_spots; wm.batch_hi = &h->d_seq->batch;
    ScoreArgs sa{};
    sa.edep = h->edep.as<float>(); sa.nvox = (unsigned long long)h->ncell; sa.sg = score_geom(h);
    const int gv = grid_for(h->ncell, h->n_sm);

    // the graph: one WHILE node whose body is the batch pass
    CU(h, cudaGraphCreate(&h->seq_graph, 0));
    cudaGraphConditionalHandle handle;
    CU(h, cudaGraphConditionalHandleCreate(&handle, h->seq_graph, 1, cudaGraphCondAssignDefault));
    cudaGraphNodeParams np = { cudaGraphNodeTypeConditional };
    np.conditional.handle = handle;
    np.conditional.type = cudaGraphCondTypeWhile;
    np.conditional.size = 1;
    cudaGraphNode_t node;
    CU(h, cudaGraphAddNode(&node, h->seq_graph, nullptr, 0, &np));
    cudaGraph_t body = np.conditional.phGraph_out[0];
    CU(h, cudaStreamBeginCaptureToGraph(st, body, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed));
    enqueue_chunk<0>(h, c, wm, 0ull, cb, sa, h->d_tal, st, false);
    seq_accumulate_kernel<<<gv, 256, 0, st>>>(h->edep.as<float>(), h->d_s1, h->d_s2, h->ncell, h->d_seq);
    seq_uncertainty_kernel<<<gv, 256, 0, st>>>(h->d_s1, h->d_s2, h->ncell, h->d_seq);
    seq_decide_kernel<<<1, 1, 0, st>>>(handle, h->d_seq, (int)min_batches, (int)max_batches, target_rel_unc);
    cudaError_t ce = cudaStreamEndCapture(st, nullptr);
    if (ce != cudaSuccess) { cudaGetLastError(); seq_release(h); FAIL(h, VPMC_ERR_CUDA, "graph capture of the batch pass: %s", cudaGetErrorString(ce)); }
    CU(h, cudaGraphInstantiate(&h->seq_exec, h->seq_graph, 0));
    CU(h, cudaGraphLaunch(h->seq_exec, st));
    double W = 0.0;
    for (double x : h->spot_w) W += x;
    const double V = (double)h->G.hx * h->G.hy * h->G.hz * 1e-3;
    const float coef_batch = (float)(W / (double)batch_histories / V * 1.602176634e-10);
    seq_finalize_kernel<<<gv, 256, 0, st>>>(h->d_s1, h->d_hu, h->d_lut, h->G, h->params.rho_min, coef_batch, h->d_seq, dose_out_dev, h->ncell, h->d_cell_rho);
    CU(h, cudaGetLastError());
    CU(h, cudaEventRecord(h->seq_ev_out, st));
    CU(h, cudaStreamWaitEvent(caller, h->seq_ev_out, 0));
    h->seq_valid = true;
    return VPMC_OK;
}

extern "C" int vpmc_get_run_info(vpmc_t *h, int32_t *batches_out, float *rel_unc_out, int32_t *reached_target_out)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    if (!h->seq_valid) FAIL(h, VPMC_ERR_STATE, "no vpmc_dose_to_uncertainty run yet");
    CU(h, cudaStreamSynchronize(h->seq_stream));
    SeqState s;
    CU(h, cudaMemcpy(&s, h->d_seq, sizeof(s), cudaMemcpyDeviceToHost));
    if (h->seq_exec) { h->launches += (unsigned long long)(chunk_launches(h) + 3u) * s.batch + 1ull; seq_release(h); }     // counted once, when the result is read
    if (batches_out) *batches_out = (int32_t)s.batch;
    if (rel_unc_out) *rel_unc_out = s.unc;
    if (reached_target_out) *reached_target_out = (int32_t)s.stopped_by_target;
    return VPMC_OK;
}

extern "C" int vpmc_get_tallies(vpmc_t *h, vpmc_tallies *out)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    if (!out) FAIL(h, VPMC_ERR_INVALID_ARG, "NULL argument");
    static_assert(sizeof(DevTallies) == sizeof(vpmc_tallies), "tally layout");
    CU(h, cudaStreamSynchronize(h->last_stream));
    CU(h, cudaMemcpy(out, h->d_tal, sizeof(DevTallies), cudaMemcpyDeviceToHost));
    return VPMC_OK;
}

extern "C" int vpmc_get_uncertainty(vpmc_t *h, float *rel_unc_out)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    if (!rel_unc_out) FAIL(h, VPMC_ERR_INVALID_ARG, "NULL argument");
    if (!h->unc_valid) FAIL(h, VPMC_ERR_STATE, "no dose run with n_batches >= 2 yet");
    double acc[2];
    CU(h, cudaStreamSynchronize(h->last_stream));
    CU(h, cudaMemcpy(acc, h->d_unc, sizeof(acc), cudaMemcpyDeviceToHost));
    *rel_unc_out = acc[1] > 0 ? (float)(acc[0] / acc[1]) : 0.0f;
    return VPMC_OK;
}

extern "C" int vpmc_trace(vpmc_t *h, const vpmc_scenario *scp, int32_t mode, uint64_t n_or_hps, uint64_t seed,
                          const uint64_t *hids, int32_t n, int32_t max_steps, vpmc_step_rec *out_host, int32_t *nrec_host)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    if (!hids || !out_host || !nrec_host || n < 0 || max_steps < 1 || n_or_hps == 0) FAIL(h, VPMC_ERR_INVALID_ARG, "bad trace arguments");
    static_assert(sizeof(StepRec) == sizeof(vpmc_step_rec), "step record layout");
    const vpmc_scenario sc = scp ? *scp : vpmc_scenario{ { 0, 0, 0 }, 1.0f };
    int rc = prepare_beams(h, sc, nullptr); if (rc) return rc;
    if (n == 0) return VPMC_OK;
    std::vector<int> spot_of(n, -1);
    if (mode == 0) {
        std::vector<unsigned long long> cnt, start(h->n_spots + 1, 0ull);
        apportion(n_or_hps, h->spot_w, cnt);
        for (int g = 0; g < h->n_spots; ++g) start[g + 1] = start[g] + cnt[g];
        for (int i = 0; i < n; ++i) {
            if (hids[i] >= n_or_hps) continue;
            const int g = (int)(std::upper_bound(start.begin(), start.end(), (unsigned long long)hids[i]) - start.begin()) - 1;
            spot_of[i] = g;
        }
    } else {
        for (int i = 0; i < n; ++i) {
            const unsigned long long g = hids[i] / n_or_hps;
            if (g < (unsigned long long)h->n_spots) spot_of[i] = (int)g;
        }
    }
    unsigned long long *d_h = nullptr; int *d_s = nullptr, *d_n = nullptr; StepRec *d_r = nullptr;
    cudaError_t e = cudaSuccess;
    auto cleanup = [&]() { cudaFree(d_h); cudaFree(d_s); cudaFree(d_n); cudaFree(d_r); };
#define CT_(x) do { e = (x); if (e != cudaSuccess) { cleanup(); FAIL(h, VPMC_ERR_CUDA, "%s: %s", #x, cudaGetErrorString(e)); } } while (0)
    CT_(cudaMalloc(&d_h, n * sizeof(unsigned long long)));
    CT_(cudaMalloc(&d_s, n * sizeof(int)));
    CT_(cudaMalloc(&d_n, n * sizeof(int)));
    CT_(cudaMalloc(&d_r, (size_t)n * max_steps * sizeof(StepRec)));
    CT_(cudaMemcpy(d_h, hids, n * sizeof(unsigned long long), cudaMemcpyHostToDevice));
    CT_(cudaMemcpy(d_s, spot_of.data(), n * sizeof(int), cudaMemcpyHostToDevice));
    CT_(cudaMemset(d_r, 0, (size_t)n * max_steps * sizeof(StepRec)));
    trace_kernel<<<(n + 63) / 64, 64>>>(make_ctx(h, sc, seed), d_h, d_s, n, h->d_spots, h->d_spot_R0, h->d_spot_beam, h->d_lut, d_r, max_steps, d_n);
    CT_(cudaGetLastError());
    h->launches += 1;
    CT_(cudaDeviceSynchronize());
    CT_(cudaMemcpy(out_host, d_r, (size_t)n * max_steps * sizeof(StepRec), cudaMemcpyDeviceToHost));
    CT_(cudaMemcpy(nrec_host, d_n, n * sizeof(int), cudaMemcpyDeviceToHost));
#undef CT_
    cleanup();
    return VPMC_OK;
}

extern "C" int vpmc_digests(vpmc_t *h, const vpmc_scenario *scp, uint64_t n_histories, uint64_t seed, uint64_t hid_begin, int32_t n,
                            vpmc_digest *out_host)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    if (n < 0 || (n > 0 && !out_host) || hid_begin + (uint64_t)n > n_histories) FAIL(h, VPMC_ERR_INVALID_ARG, "bad digest arguments");
    static_assert(sizeof(Digest) == sizeof(vpmc_digest), "digest layout");
    const vpmc_scenario sc = scp ? *scp : vpmc_scenario{ { 0, 0, 0 }, 1.0f };
    int rc = prepare_beams(h, sc, nullptr); if (rc) return rc;
    if (n == 0) return VPMC_OK;
    std::vector<unsigned long long> cnt, start(h->n_spots + 1, 0ull);
    apportion(n_histories, h->spot_w, cnt);
    for (int g = 0; g < h->n_spots; ++g) start[g + 1] = start[g] + cnt[g];
    DevBuf dstart, dout;
    if ((rc = ensure(h, dstart, start.size() * sizeof(unsigned long long))) || (rc = ensure(h, dout, (size_t)n * sizeof(Digest)))) { pool_give(dstart.p, dstart.bytes); return rc; }
    cudaError_t e = cudaMemcpy(dstart.p, start.data(), start.size() * sizeof(unsigned long long), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        digest_kernel<<<(n + 63) / 64, 64>>>(make_ctx(h, sc, seed), hid_begin, n, dstart.as<unsigned long long>(), h->n_spots, h->d_spots, h->d_spot_R0,
                                             h->d_spot_beam, h->d_lut, dout.as<Digest>());
        h->launches += 1;
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e == cudaSuccess) e = cudaMemcpy(out_host, dout.p, (size_t)n * sizeof(Digest), cudaMemcpyDeviceToHost);
    pool_give(dstart.p, dstart.bytes); pool_give(dout.p, dout.bytes);
    if (e != cudaSuccess) FAIL(h, VPMC_ERR_CUDA, "digests: %s", cudaGetErrorString(e));
    return VPMC_OK;
}

extern "C" int vpmc_step_from_state(vpmc_t *h, const vpmc_scenario *scp, uint64_t seed, const vpmc_state *states, int32_t n,
                                    vpmc_state_out *out)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    if (n < 0 || (n > 0 && (!states || !out))) FAIL(h, VPMC_ERR_INVALID_ARG, "bad step_from_state arguments");
    static_assert(sizeof(StateIn) == sizeof(vpmc_state) && sizeof(StateOut) == sizeof(vpmc_state_out), "state layout");
    const vpmc_scenario sc = scp ? *scp : vpmc_scenario{ { 0, 0, 0 }, 1.0f };
    int rc = prepare_beams(h, sc, nullptr); if (rc) return rc;
    if (n == 0) return VPMC_OK;
    for (int i = 0; i < n; ++i) {
        const vpmc_state &q = states[i];
        if (q.kind < VPMC_STEP_SOURCE || q.kind > VPMC_STEP_CT || q.beam < 0 || q.beam >= (int)h->beams.size()) FAIL(h, VPMC_ERR_INVALID_ARG, "state %d: bad kind or beam", i);
        if (q.kind == VPMC_STEP_SOURCE && (q.spot < 0 || q.spot >= h->n_spots || h->spot_beam_h[q.spot] != q.beam)) FAIL(h, VPMC_ERR_INVALID_ARG, "state %d: bad spot", i);
        if (q.kind == VPMC_STEP_CT)
            for (int a = 0; a < 3; ++a)
                if (q.ivox[a] < 0 || q.ivox[a] >= (a == 0 ? h->G.nx : a == 1 ? h->G.ny : h->G.nz)) FAIL(h, VPMC_ERR_INVALID_ARG, "state %d: voxel outside the grid", i);
        const BeamHost &b = h->beams[q.beam];
        if (((q.kind == VPMC_STEP_DRIFT_TO_RS || q.kind == VPMC_STEP_RS) && !(b.rs_wet > 0.0f)) ||
            ((q.kind == VPMC_STEP_DRIFT_TO_AP || q.kind == VPMC_STEP_AP) && !b.has_ap)) FAIL(h, VPMC_ERR_INVALID_ARG, "state %d: the beam has no such device", i);
    }
    DevBuf din, dout;
    if ((rc = ensure(h, din, (size_t)n * sizeof(StateIn))) || (rc = ensure(h, dout, (size_t)n * sizeof(StateOut)))) { pool_give(din.p, din.bytes); return rc; }
    cudaError_t e = cudaMemcpy(din.p, states, (size_t)n * sizeof(StateIn), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        step_state_kernel<<<(n + 63) / 64, 64>>>(make_ctx(h, sc, seed), din.as<StateIn>(), n, h->d_spots, h->d_spot_R0, h->d_lut, dout.as<StateOut>());
        h->launches += 1;
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e == cudaSuccess) e = cudaMemcpy(out, dout.p, (size_t)n * sizeof(StateOut), cudaMemcpyDeviceToHost);
    pool_give(din.p, din.bytes); pool_give(dout.p, dout.bytes);
    if (e != cudaSuccess) FAIL(h, VPMC_ERR_CUDA, "step_from_state: %s", cudaGetErrorString(e));
    return VPMC_OK;
}

#include "vpmc_influence.inl"
#include "vpmc_spmv.inl"
