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
        if (h->d_spots) cudaFree(h->d_spots);
        if (h->d_spot_R0) cudaFree(h->d_spot_R0);
        h->d_spot_R0 = nullptr;
        if (h->d_spot_beam) cudaFree(h->d_spot_beam);
        if (h->d_beams) cudaFree(h->d_beams);
        h->d_spots = nullptr; h->d_spot_beam = nullptr; h->d_beams = nullptr;
        CU(h, cudaMalloc(&h->d_spots, sp.size() * sizeof(float4)));
        CU(h, cudaMalloc(&h->d_spot_beam, sp.size() * sizeof(int)));
        CU(h, cudaMalloc(&h->d_beams, h->beams.size() * sizeof(DevBeam)));
        CU(h, cudaMemcpy(h->d_spots, sp.data(), sp.size() * sizeof(float4), cudaMemcpyHostToDevice));
        CU(h, cudaMalloc(&h->d_spot_R0, r0.size() * sizeof(double)));
        CU(h, cudaMemcpy(h->d_spot_R0, r0.data(), r0.size() * sizeof(double), cudaMemcpyHostToDevice));
        CU(h, cudaMemcpy(h->d_spot_beam, h->spot_beam_h.data(), sp.size() * sizeof(int), cudaMemcpyHostToDevice));
        if (h->map_capacity < h->n_spots + 1) {
            if (h->d_cum) cudaFree(h->d_cum);
            if (h->d_first) cudaFree(h->d_first);
            h->d_cum = nullptr; h->d_first = nullptr;
            CU(h, cudaMalloc(&h->d_cum, ((size_t)h->n_spots + 1) * sizeof(unsigned long long)));
            CU(h, cudaMalloc(&h->d_first, ((size_t)h->n_spots + 1) * sizeof(unsigned long long)));
            h->map_capacity = h->n_spots + 1;
        }
        h->spots_dirty = false;
    }
    std::vector<DevBeam> db(h->beams.size());
    for (size_t i = 0; i < h->beams.size(); ++i) {
        const BeamHost &b = h->beams[i];
        DevBeam &d = db[i];
        memcpy(d.iso, b.frame.iso, sizeof(d.iso));
        memcpy(d.rot, b.frame.rot, sizeof(d.rot));
        d.has_rs = b.rs_wet > 0.0f;
        d.w_rs_out = -b.rs_face;
        d.w_rs_in = d.w_rs_out - b.rs_wet / h->params.rs_rsp;
        d.has_ap = b.has_ap;
        d.w_ap_out = -b.ap_face;
        d.w_ap_in = d.w_ap_out - b.ap_T;
        d.ap_bits = b.d_bits; d.ap_nx = b.ap_nx; d.ap_ny = b.ap_ny; d.ap_row_words = b.ap_row_words;
        d.ap_u0 = b.ap_u0; d.ap_v0 = b.ap_v0; d.ap_du = b.ap_du; d.ap_dv = b.ap_dv;
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

// one chunk: beam line for `n` items starting at item0, then the persistent voxel kernel on the survivors
template <int MODE>
static int launch_chunk(vpmc_t *h, const WorkMap &wm0, unsigned long long item0, unsigned int n, const vpmc_scenario &sc,
                        uint64_t seed, float *edep, const ColumnBoxes &cb, int col0, cudaStream_t st)
{
    WorkMap wm = wm0;
    wm.item0 = item0; wm.n_items = n;
    CU(h, cudaMemsetAsync(h->d_qctr, 0, 2 * sizeof(unsigned int), st));
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    const float3 shift = make_float3(sc.shift[0], sc.shift[1], sc.shift[2]);
    {
        TimedScope ts(h, st, 0);
        beamline_kernel<<<(n + 255) / 256, 256, 0, st>>>(h->P, h->G, wm, h->d_spots, h->d_spot_R0, h->d_spot_beam, h->d_beams, shift, k0, k1, h->q, h->d_tal);
    }
    CU(h, cudaGetLastError());
    TimedScope ts(h, st, 1);
    if (h->smem_lut)
        voxel_kernel<MODE, true><<<h->voxel_grid[MODE][1], 256, h->lut_bytes, st>>>(h->P, h->G, h->q, h->d_hu, h->d_lut, sc.rsp_scale, edep, cb, col0, wm.hps, k0, k1, h->d_tal);
    else
        voxel_kernel<MODE, false><<<h->voxel_grid[MODE][0], 256, 0, st>>>(h->P, h->G, h->q, h->d_hu, h->d_lut, sc.rsp_scale, edep, cb, col0, wm.hps, k0, k1, h->d_tal);
    CU(h, cudaGetLastError());
    h->launches += 2;
    return VPMC_OK;
}

static int grid_for(long long n, int n_sm) { return (int)std::min<long long>((n + 255) / 256, (long long)n_sm * 16); }

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
        CU(h, cudaMalloc(&h->d_s1, h->nvox * sizeof(float)));
        CU(h, cudaMalloc(&h->d_s2, h->nvox * sizeof(float)));
    }
    // C2: history ids are contiguous per spot in spot order
    std::vector<unsigned long long> cnt, start(h->n_spots + 1, 0ull);
    apportion(n_histories, h->spot_w, cnt);
    for (int g = 0; g < h->n_spots; ++g) start[g + 1] = start[g] + cnt[g];
    const unsigned long long wlo = h->win_lo, whi = h->win_hi ? std::min<unsigned long long>(h->win_hi, n_histories) : n_histories;

    CU(h, cudaMemsetAsync(h->d_edep, 0, h->nvox * sizeof(float), st));
    CU(h, cudaMemsetAsync(h->d_sum, 0, h->nvox * sizeof(float), st));
    if (with_unc) {
        CU(h, cudaMemsetAsync(h->d_s1, 0, h->nvox * sizeof(float), st));
        CU(h, cudaMemsetAsync(h->d_s2, 0, h->nvox * sizeof(float), st));
    }
    CU(h, cudaMemsetAsync(h->d_tal, 0, sizeof(DevTallies), st));
    CU(h, cudaMemsetAsync(h->d_max_bits, 0, sizeof(unsigned int), st));
    CU(h, cudaMemsetAsync(h->d_unc, 0, 2 * sizeof(double), st));

    // total items in the window (for the batch scale factor)
    std::vector<std::vector<unsigned long long>> cum(B), first(B);
    unsigned long long n_total = 0;
    for (int b = 0; b < B; ++b) {
        cum[b].assign(h->n_spots + 1, 0ull); first[b].assign(h->n_spots + 1, 0ull);
        for (int g = 0; g < h->n_spots; ++g) {
            const unsigned __int128 n = cnt[g];
            unsigned long long lo = start[g] + (unsigned long long)((n * (unsigned)b) / (unsigned)B);
            unsigned long long hi = start[g] + (unsigned long long)((n * (unsigned)(b + 1)) / (unsigned)B);
            lo = std::max(lo, wlo); hi = std::min(hi, whi);
            first[b][g] = lo;
            cum[b][g + 1] = cum[b][g] + (hi > lo ? hi - lo : 0ull);
        }
        n_total += cum[b][h->n_spots];
    }
    ColumnBoxes cb{};
    for (int b = 0; b < B; ++b) {
        const unsigned long long nb = cum[b][h->n_spots];
        if (nb == 0) continue;
        CU(h, cudaMemcpyAsync(h->d_cum, cum[b].data(), ((size_t)h->n_spots + 1) * sizeof(unsigned long long), cudaMemcpyHostToDevice, st));
        CU(h, cudaMemcpyAsync(h->d_first, first[b].data(), ((size_t)h->n_spots + 1) * sizeof(unsigned long long), cudaMemcpyHostToDevice, st));
        WorkMap wm{};
        wm.mode = 0; wm.cum = h->d_cum; wm.first = h->d_first; wm.n_spots = h->n_spots;
        for (unsigned long long i0 = 0; i0 < nb; i0 += kChunk) {
            const unsigned int n = (unsigned int)std::min<unsigned long long>(kChunk, nb - i0);
            rc = launch_chunk<0>(h, wm, i0, n, sc, seed, h->d_edep, cb, 0, st); if (rc) return rc;
        }
        const float f = (float)((double)n_total / (double)nb);
        TimedScope ts(h, st, 2);
        batch_accumulate_kernel<<<grid_for(h->nvox, h->n_sm), 256, 0, st>>>(h->d_edep, h->d_sum, h->d_s1, h->d_s2, h->nvox, f, with_unc ? 1 : 0);
        CU(h, cudaGetLastError());
        h->launches += 1;
    }
    // C6
    double W = 0.0;
    for (double x : h->spot_w) W += x;
    const double V = (double)h->G.hx * h->G.hy * h->G.hz * 1e-3;
    const float coef = (float)((n_histories ? W / (double)n_histories : 0.0) / V * 1.602176634e-10);
    TimedScope ts(h, st, 2);
    dose_convert_kernel<<<grid_for(h->nvox, h->n_sm), 256, 0, st>>>(h->d_sum, h->d_hu, h->d_lut, h->G, h->params.rho_min, coef, dose_out_dev, h->nvox, h->d_max_bits);
    CU(h, cudaGetLastError());
    h->launches += 1;
    if (with_unc) {
        uncertainty_kernel<<<grid_for(h->nvox, h->n_sm), 256, 0, st>>>(dose_out_dev, h->d_s1, h->d_s2, h->nvox, B, h->d_max_bits, h->d_unc);
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
    float *d = nullptr;
    CU(h, cudaMalloc(&d, h->nvox * sizeof(float)));
    int rc = vpmc_dose(h, n_histories, seed, d, nullptr);
    if (rc == VPMC_OK) {
        cudaError_t e = cudaMemcpy(dose_out_host, d, h->nvox * sizeof(float), cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) { h->err = cudaGetErrorString(e); rc = VPMC_ERR_CUDA; }
    }
    cudaFree(d);
    return rc;
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
    trace_kernel<true><<<(n + 63) / 64, 64>>>(h->P, h->G, d_h, d_s, n, h->d_spots, h->d_spot_R0, h->d_spot_beam, h->d_beams,
                                             make_float3(sc.shift[0], sc.shift[1], sc.shift[2]), h->d_hu, h->d_lut, sc.rsp_scale,
                                             (uint32_t)seed, (uint32_t)(seed >> 32), d_r, max_steps, d_n);
    CT_(cudaGetLastError());
    h->launches += 1;
    CT_(cudaDeviceSynchronize());
    CT_(cudaMemcpy(out_host, d_r, (size_t)n * max_steps * sizeof(StepRec), cudaMemcpyDeviceToHost));
    CT_(cudaMemcpy(nrec_host, d_n, n * sizeof(int), cudaMemcpyDeviceToHost));
#undef CT_
    cleanup();
    return VPMC_OK;
}

#include "vpmc_influence.inl"
