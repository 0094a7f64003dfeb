// vpmc_api.cu -- the C-ABI of libvpmc.so (include/vpmc.h): host set-up (S0) and launch sequencing.
// Every step of the hot path runs in the kernels of vpmc_kernels.cuh; there is no CPU fallback.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <mutex>
#include <numeric>

#include "vpmc_host.h"
#include "vpmc_setup.cuh"

using namespace vpk;

static thread_local std::string g_create_err;

#define FAIL(h, code, ...)                                      \
    do {                                                        \
        char _b[512];                                           \
        snprintf(_b, sizeof(_b), __VA_ARGS__);                  \
        if (h) (h)->err = _b; else g_create_err = _b;           \
        return (code);                                          \
    } while (0)

#define CU(h, expr)                                                                         \
    do {                                                                                    \
        cudaError_t _e = (expr);                                                            \
        if (_e != cudaSuccess) FAIL(h, VPMC_ERR_CUDA, "%s: %s", #expr, cudaGetErrorString(_e)); \
    } while (0)

static constexpr size_t kMaxSmemLut = 16 * 1024;      // larger material tables are read through L1 instead: a 64 KB table in
                                                      // shared memory costs the voxel kernel its fourth CTA per SM (measured +1-2.5 %)

// ---- vpmc_spmv_grad_static: the one entry point that allocates nothing (include/vpmc.h).  Its scratch -- the first / last
// partial sums per chunk of spmv_grad_kernel -- lives in this file-scope device array: 2 floats per chunk of kSpmvChunk entries,
// VPMC_STATIC_MAX_NNZ entries at most = 256 KB, held by every GPU that loads the library until the process exits.  In host
// code the NAME of the array is a host-side stand-in, not a device address: static_scratch_for_device() asks the runtime for
// the address once per device (with that device current) and the launches are given that pointer.
static_assert(VPMC_STATIC_MAX_NNZ % kSpmvChunk == 0, "the static scratch is sized in whole chunks");
constexpr int kStaticChunks = (int)(VPMC_STATIC_MAX_NNZ / kSpmvChunk);
static __device__ __align__(256) float g_spmv_static_part[2 * kStaticChunks];

namespace {
constexpr int kMaxDevices = 64;
std::mutex g_static_mu;
float *g_static_ptr[kMaxDevices] = {};
bool g_static_tried[kMaxDevices] = {};
std::string g_static_err[kMaxDevices];

// device address of g_spmv_static_part on the CURRENT device `dev` (looked up once per device); NULL + *err on failure
float *static_scratch_for_device(int dev, std::string *err)
{
    if (dev < 0 || dev >= kMaxDevices) { if (err) *err = "device index beyond the static-scratch table"; return nullptr; }
    std::lock_guard<std::mutex> lk(g_static_mu);
    if (!g_static_tried[dev]) {
        g_static_tried[dev] = true;
        void *ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&ptr, g_spmv_static_part);
        if (e != cudaSuccess) { cudaGetLastError(); g_static_err[dev] = std::string("cudaGetSymbolAddress(g_spmv_static_part): ") + cudaGetErrorString(e); }
        else g_static_ptr[dev] = static_cast<float *>(ptr);
    }
    if (!g_static_ptr[dev] && err) *err = g_static_err[dev];
    return g_static_ptr[dev];
}
}  // namespace

// grow-only device buffer
static int ensure(vpmc_t *h, DevBuf &b, size_t bytes);

// Process-wide cache of released device buffers: engines are created and destroyed per plan (bench.py's e2e leg does
// exactly that), and cudaMalloc / cudaFree of the ~1 GB of record queues would otherwise dominate a 10 ms dose.
namespace {
struct PoolEntry { void *p; size_t bytes; int device; };
std::mutex g_pool_mu;
std::vector<PoolEntry> g_pool;
size_t g_pool_bytes = 0;
constexpr size_t kPoolLimit = (size_t)16 << 30;

int current_device() { int d = 0; cudaGetDevice(&d); return d; }

void *pool_take(size_t want, size_t &got)
{
    const int dev = current_device();
    std::lock_guard<std::mutex> lk(g_pool_mu);
    // best fit; a buffer of up to 16x the size asked for is still better than a cudaMalloc (tens of ms for the record
    // queues of a plan whose beam line differs from the previous plans')
    int best = -1;
    for (int i = 0; i < (int)g_pool.size(); ++i)
        if (g_pool[i].device == dev && g_pool[i].bytes >= want && g_pool[i].bytes <= 16 * want + 4096 && (best < 0 || g_pool[i].bytes < g_pool[best].bytes)) best = i;
    if (best < 0) return nullptr;
    void *p = g_pool[best].p; got = g_pool[best].bytes;
    g_pool_bytes -= got;
    g_pool.erase(g_pool.begin() + best);
    return p;
}

void pool_give(void *p, size_t bytes)
{
    if (!p) return;
    {
        const int dev = current_device();
        std::lock_guard<std::mutex> lk(g_pool_mu);
        if (g_pool_bytes + bytes <= kPoolLimit && g_pool.size() < 2048) { g_pool.push_back({ p, bytes, dev }); g_pool_bytes += bytes; return; }
    }
    cudaFree(p);
}
}  // namespace

static int ensure(vpmc_t *h, DevBuf &b, size_t bytes)
{
    if (b.bytes >= bytes && b.p) return VPMC_OK;
    if (b.p) { cudaDeviceSynchronize(); pool_give(b.p, b.bytes); b.p = nullptr; b.bytes = 0; }   // rare: growth of a live buffer
    const size_t want = std::max<size_t>(bytes, 256);
    size_t got = 0;
    if (void *p = pool_take(want, got)) { b.p = p; b.bytes = got; return VPMC_OK; }
    if (cudaMalloc(&b.p, want) != cudaSuccess) {
        cudaGetLastError(); b.p = nullptr;
        // the cache may be holding what is missing: drop it and retry once
        { std::lock_guard<std::mutex> lk(g_pool_mu); for (auto &e : g_pool) cudaFree(e.p); g_pool.clear(); g_pool_bytes = 0; }
        if (cudaMalloc(&b.p, want) != cudaSuccess) { cudaGetLastError(); b.p = nullptr; FAIL(h, VPMC_ERR_ALLOC, "out of device memory (%zu bytes)", want); }
    }
    b.bytes = want;
    return VPMC_OK;
}

// fixed-size device members of a handle: taken from the buffer cache, remembered in h->owned, returned in vpmc_destroy
static int dev_alloc(vpmc_t *h, void **out, size_t bytes)
{
    DevBuf b;
    int rc = ensure(h, b, bytes); if (rc) { *out = nullptr; return rc; }
    h->owned.push_back({ b.p, b.bytes });
    *out = b.p;
    return VPMC_OK;
}

// give one member back while the handle lives on (inputs replaced by a later set_* call): whatever may still read it must
// have finished first
static void dev_release(vpmc_t *h, void *p)
{
    if (!p) return;
    for (size_t i = 0; i < h->owned.size(); ++i)
        if (h->owned[i].p == p) {
            if (h->launched) cudaStreamSynchronize(h->last_stream);
            if (h->setup_stream) cudaStreamSynchronize(h->setup_stream);
            pool_give(p, h->owned[i].bytes);
            h->owned.erase(h->owned.begin() + i);
            return;
        }
}

// the stream of a compute call waits for the set-up work enqueued so far
static void join_setup(vpmc_t *h, cudaStream_t st)
{
    if (!h->setup_pending) return;
    cudaEventRecord(h->setup_ev, h->setup_stream);
    cudaStreamWaitEvent(st, h->setup_ev, 0);
    h->setup_pending = false;
}

extern "C" const char *vpmc_version(void) { return "vpmc-b200 0.2 (sm_100a)"; }

extern "C" void vpmc_default_params(vpmc_params *p)
{
    if (!p) return;
    p->alpha = 0.022f; p->p = 1.77f; p->X0_w = 360.8f; p->Es = 13.6f; p->c_log = 0.038f;
    p->beta_nuc = 0.0012f; p->gamma_loc = 0.6f; p->k_bohr = 0.015692f; p->za_w = 0.5551f;
    p->R_cut = 0.1f; p->f_R = 0.25f; p->s_max = std::numeric_limits<float>::infinity(); p->s_rs = 1.0f; p->s_ap = 1.0f;
    p->brass_rsp = 5.523f; p->brass_rho = 8.5f; p->brass_X0 = 14.94f; p->brass_za = 0.457f;
    p->rs_rsp = 1.0f; p->rs_rho = 1.0f; p->rs_X0 = 360.8f;
    p->rho_min = 1e-3f; p->delta_E = 0.0f;
    p->flags = VPMC_FLAG_MCS | VPMC_FLAG_STRAGGLE | VPMC_FLAG_NUCLEAR;
    p->n_batches = 10;
}

static DevParams make_dev_params(const vpmc_params &p)
{
    DevParams d;
    d.alpha = p.alpha; d.p = p.p; d.inv_p = (float)(1.0 / (double)p.p); d.inv_alpha = (float)(1.0 / (double)p.alpha);
    d.inv_X0_w = (float)(1.0 / (double)p.X0_w); d.Es = p.Es; d.c_log = p.c_log;
    d.beta_nuc = p.beta_nuc; d.gamma_loc = p.gamma_loc; d.k_bohr = p.k_bohr; d.za_w = p.za_w;
    d.R_cut = p.R_cut; d.f_R = p.f_R; d.s_max = p.s_max; d.s_rs = p.s_rs; d.s_ap = p.s_ap;
    d.brass_rsp = p.brass_rsp; d.brass_inv_rsp = (float)(1.0 / (double)p.brass_rsp); d.brass_rho = p.brass_rho;
    d.brass_inv_X0 = (float)(1.0 / (double)p.brass_X0);
    d.brass_za_rho = (float)((double)p.brass_za * (double)p.brass_rho);
    d.rs_rsp = p.rs_rsp; d.rs_inv_rsp = (float)(1.0 / (double)p.rs_rsp); d.rs_rho = p.rs_rho; d.rs_inv_X0 = (float)(1.0 / (double)p.rs_X0);
    d.rs_za_rho = (float)((double)p.za_w * (double)p.rs_rho);
    d.rho_min = p.rho_min; d.delta_E = p.delta_E; d.flags = p.flags; d.R_cut_d = (double)p.R_cut;
    const double pp = (double)p.p;
    d.pc2 = (float)(pp * (pp - 1) / 2); d.pc3 = (float)(pp * (pp - 1) * (pp - 2) / 6);
    d.pc4 = (float)(pp * (pp - 1) * (pp - 2) * (pp - 3) / 24); d.pc5 = (float)(pp * (pp - 1) * (pp - 2) * (pp - 3) * (pp - 4) / 120);
    return d;
}

static double pl_eval(const vpmc_calib *c, const float *y, double hu)
{
    if (hu <= c->hu[0]) return y[0];
    if (hu >= c->hu[c->n - 1]) return y[c->n - 1];
    int k = 0;
    while (k + 2 < c->n && hu >= c->hu[k + 1]) ++k;
    const double t = (hu - c->hu[k]) / ((double)c->hu[k + 1] - (double)c->hu[k]);
    return (double)y[k] + t * ((double)y[k + 1] - (double)y[k]);
}

static void free_beam(vpmc_t *h, BeamHost &b)
{
    dev_release(h, b.d_bits); dev_release(h, b.d_dist); dev_release(h, b.d_ap_tmp); dev_release(h, b.d_poly); dev_release(h, b.d_pgrid); dev_release(h, b.d_prows);
    b.d_bits = nullptr; b.d_dist = nullptr; b.d_ap_tmp = nullptr; b.d_poly = nullptr; b.d_pgrid = nullptr; b.d_prows = nullptr; b.ap_n_poly = 0;
}

extern "C" int vpmc_destroy(vpmc_t *h)
{
    if (!h) return VPMC_OK;
    // only this handle's own streams are drained (no device-wide synchronisation)
    if (h->launched) cudaStreamSynchronize(h->last_stream);
    if (h->setup_stream) cudaStreamSynchronize(h->setup_stream);
    if (h->seq_stream) cudaStreamSynchronize(h->seq_stream);
    for (auto &t : h->timed) { cudaEventDestroy(t.a); cudaEventDestroy(t.b); }
    if (h->seq_exec) cudaGraphExecDestroy(h->seq_exec);
    if (h->seq_graph) cudaGraphDestroy(h->seq_graph);
    if (h->seq_ev_in) cudaEventDestroy(h->seq_ev_in);
    if (h->seq_ev_out) cudaEventDestroy(h->seq_ev_out);
    if (h->seq_stream) cudaStreamDestroy(h->seq_stream);
    if (h->setup_ev) cudaEventDestroy(h->setup_ev);
    if (h->copy_ev) cudaEventDestroy(h->copy_ev);
    if (h->setup_stream) cudaStreamDestroy(h->setup_stream);
    for (auto &o : h->owned) pool_give(o.p, o.bytes);
    h->owned.clear();
    DevBuf *bufs[] = { &h->cum, &h->first, &h->edep, &h->s0, &h->s1, &h->s2, &h->a0, &h->a1, &h->a2, &h->a3, &h->a4, &h->b0, &h->b1, &h->b2, &h->b3, &h->b4, &h->b5, &h->q0, &h->q1, &h->q2, &h->q3, &h->q4, &h->inf_scratch, &h->inf_lo, &h->inf_dim, &h->inf_off, &h->inf_bbox, &h->inf_cols,
                       &h->inf_tile0, &h->inf_tilecol, &h->inf_skip, &h->inf_tilecnt, &h->inf_colmax, &h->inf_colnnz, &h->inf_colbase,
                       &h->inf_stage_idx, &h->inf_stage_val, &h->inf_rowsrc, &h->ovf_key, &h->ovf_val, &h->ovf_key2, &h->ovf_val2, &h->ovf_flag,
                       &h->ovf_colcnt, &h->ovf_coloff, &h->ovf_kept, &h->ovf_ctr, &h->ostage_idx, &h->ostage_val, &h->row_ovf_off, &h->row_ovf_n, &h->spmv_part, &h->gamma_buf };
    for (DevBuf *b : bufs) if (b->p) { pool_give(b->p, b->bytes); b->p = nullptr; }
    delete h;
    return VPMC_OK;
}

// the persistent kernels by (stage | mode, table placement, fl): fl = 1 is the specialisation for flags == 7
typedef void (*BeamFn)(const Ctx, const SourceBuf, const Queue, const Queue, unsigned int *, DevTallies *);
typedef void (*VoxelFn)(const Ctx, const Queue, const float4 *, const ScoreArgs, DevTallies *);
static BeamFn beam_fn(int stage, int fl)
{
    static const BeamFn t[2][2] = { { beam_kernel<0, -1>, beam_kernel<0, 7> }, { beam_kernel<1, -1>, beam_kernel<1, 7> } };
    return t[stage][fl];
}
static VoxelFn voxel_fn(int mode, int smem, int fl)
{
    static const VoxelFn t[3][2][2] = { { { voxel_kernel<0, false, -1>, voxel_kernel<0, false, 7> }, { voxel_kernel<0, true, -1>, voxel_kernel<0, true, 7> } },
                                        { { voxel_kernel<1, false, -1>, voxel_kernel<1, false, 7> }, { voxel_kernel<1, true, -1>, voxel_kernel<1, true, 7> } },
                                        { { voxel_kernel<2, false, -1>, voxel_kernel<2, false, 7> }, { voxel_kernel<2, true, -1>, voxel_kernel<2, true, 7> } } };
    return t[mode][smem][fl];
}

extern "C" int vpmc_create(vpmc_t **out, const vpmc_ct *ct, const vpmc_calib *cal, const vpmc_params *params)
{
    if (!out) { g_create_err = "out is NULL"; return VPMC_ERR_INVALID_ARG; }
    *out = nullptr;
    vpmc_t *nh = nullptr;
    if (!ct || !cal || !ct->hu) FAIL(nh, VPMC_ERR_INVALID_ARG, "ct / calibration missing");
    for (int a = 0; a < 3; ++a)
        if (ct->n[a] < 1 || ct->n[a] > 65535 || !(ct->h[a] > 0.0f)) FAIL(nh, VPMC_ERR_INVALID_ARG, "bad CT grid on axis %d", a);
    const long long nvox = (long long)ct->n[0] * ct->n[1] * ct->n[2];
    if (nvox > 0x7fffffffLL) FAIL(nh, VPMC_ERR_INVALID_ARG, "more than 2^31-1 voxels");
    if (cal->n < 1 || !cal->hu || !cal->rsp || !cal->rho) FAIL(nh, VPMC_ERR_INVALID_ARG, "calibration needs hu, rsp, rho nodes");
    for (int k = 1; k < cal->n; ++k)
        if (!(cal->hu[k] > cal->hu[k - 1])) FAIL(nh, VPMC_ERR_INVALID_ARG, "calibration nodes must ascend in hu");
    vpmc_params p;
    if (params) p = *params; else vpmc_default_params(&p);
    if (!(p.alpha > 0) || !(p.p > 1) || !(p.R_cut > 0) || !(p.f_R > 0 && p.f_R < 1) || !(p.s_rs > 0) || !(p.s_ap > 0) ||
        !(p.brass_rsp > 0) || !(p.rs_rsp > 0) || p.n_batches < 1 || p.n_batches > 1000)
        FAIL(nh, VPMC_ERR_INVALID_ARG, "parameter out of range");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) FAIL(nh, VPMC_ERR_CUDA, "no CUDA device (this library has no CPU path)");

    vpmc_t *h = new vpmc();
    h->params = p;
    h->P = make_dev_params(p);
    h->nvox = nvox; h->ncell = nvox;
    h->sn[0] = ct->n[0]; h->sn[1] = ct->n[1]; h->sn[2] = ct->n[2];
    cudaGetDevice(&h->device);
    cudaDeviceGetAttribute(&h->n_sm, cudaDevAttrMultiProcessorCount, h->device);
    h->static_scratch = static_scratch_for_device(h->device, &h->static_scratch_err);     // set-up of vpmc_spmv_grad_static; create does not fail on it
    DevGrid &G = h->G;
    G.nx = ct->n[0]; G.ny = ct->n[1]; G.nz = ct->n[2];
    G.hx = ct->h[0]; G.hy = ct->h[1]; G.hz = ct->h[2];
    G.ox = ct->origin[0]; G.oy = ct->origin[1]; G.oz = ct->origin[2];
    // S0: per-integer-HU material table over the span of the calibration nodes (values are constant outside)
    G.hu_min = (int)std::floor((double)cal->hu[0]);
    const int hu_max = (int)std::ceil((double)cal->hu[cal->n - 1]);
    G.n_lut = hu_max - G.hu_min + 1;
    if (G.n_lut > (1 << 20)) { delete h; FAIL(nh, VPMC_ERR_INVALID_ARG, "calibration spans more than 2^20 HU"); }
    std::vector<float4> lut((size_t)G.n_lut);
    for (int i = 0; i < G.n_lut; ++i) {
        const double hu = (double)(G.hu_min + i);
        const double rsp = pl_eval(cal, cal->rsp, hu), rho = pl_eval(cal, cal->rho, hu);
        const double xsp = cal->xsp ? pl_eval(cal, cal->xsp, hu) : rho;
        if (!(rsp > 0.0)) { delete h; FAIL(nh, VPMC_ERR_INVALID_ARG, "calibration gives RSP <= 0 at HU %d", G.hu_min + i); }
        lut[i] = make_float4((float)rsp, (float)rho, (float)(xsp / (double)p.X0_w), (float)(1.0 / rsp));
    }
    h->lut_bytes = lut.size() * sizeof(float4);
    h->smem_lut = h->lut_bytes <= kMaxSmemLut;
#define CUC(expr) do { cudaError_t _e = (expr); if (_e != cudaSuccess) { g_create_err = std::string(#expr) + ": " + cudaGetErrorString(_e); vpmc_destroy(h); return VPMC_ERR_CUDA; } } while (0)
#define CUA(ptr, bytes) do { if (dev_alloc(h, (void **)&(ptr), (bytes)) != VPMC_OK) { g_create_err = h->err; vpmc_destroy(h); return VPMC_ERR_ALLOC; } } while (0)
    CUC(cudaStreamCreateWithFlags(&h->setup_stream, cudaStreamNonBlocking));
    CUC(cudaEventCreateWithFlags(&h->setup_ev, cudaEventDisableTiming));
    CUC(cudaEventCreateWithFlags(&h->copy_ev, cudaEventDisableTiming));
    cudaStream_t ss = h->setup_stream;
    CUA(h->d_lut, h->lut_bytes);
    CUA(h->d_hu, nvox * sizeof(short));
    CUA(h->d_tal, sizeof(DevTallies));
    CUA(h->d_tal_scratch, sizeof(DevTallies));
    CUA(h->d_max_bits, sizeof(unsigned int));
    CUA(h->d_unc, 2 * sizeof(double));
    CUA(h->d_qctr, 8 * sizeof(unsigned int));
    CUA(h->d_fb, 1024 * sizeof(float));
    CUC(cudaMemcpyAsync(h->d_lut, lut.data(), h->lut_bytes, cudaMemcpyHostToDevice, ss));
    CUC(cudaMemcpyAsync(h->d_hu, ct->hu, nvox * sizeof(short), ct->hu_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, ss));
    CUC(cudaMemsetAsync(h->d_tal, 0, sizeof(DevTallies), ss));
    CUC(cudaEventRecord(h->copy_ev, ss));
    h->setup_pending = true;
    // persistent kernels: one wave of resident CTAs each
    {
        h->tally_smem = (kWarps * sizeof(WarpTally) + 15) / 16 * 16;
        // occupancy queries are ~0.3 ms each: remember the answer per (device, table size, table placement)
        struct GridCache { int device; size_t lut_bytes; bool smem; int grid_beam[2][2]; int grid[3][2][2]; };
        static std::mutex mu;
        static std::vector<GridCache> cache;
        bool hit = false;
        {
            std::lock_guard<std::mutex> lk(mu);
            for (const GridCache &g : cache)
                if (g.device == h->device && g.lut_bytes == h->lut_bytes && g.smem == h->smem_lut) { memcpy(h->grid_beam, g.grid_beam, sizeof(h->grid_beam)); memcpy(h->grid, g.grid, sizeof(h->grid)); hit = true; }
        }
        if (!hit) {
            int occ = 0;
            for (int st = 0; st < 2; ++st)
                for (int f = 0; f < 2; ++f) {
                    CUC(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, beam_fn(st, f), kBlock, 0));
                    h->grid_beam[st][f] = std::max(occ, 1) * h->n_sm;
                }
            for (int m = 0; m < 3; ++m)
                for (int s = 0; s < 2; ++s)
                    for (int f = 0; f < 2; ++f) {
                        if (s == 1 && !h->smem_lut) continue;
                        const size_t sm = h->tally_smem + (s ? h->lut_bytes : 0);
                        if (s) CUC(cudaFuncSetAttribute(voxel_fn(m, s, f), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(kMaxSmemLut + h->tally_smem)));
                        CUC(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, voxel_fn(m, s, f), kBlock, sm));
                        h->grid[m][s][f] = std::max(occ, 1) * h->n_sm;
                    }
            GridCache g; g.device = h->device; g.lut_bytes = h->lut_bytes; g.smem = h->smem_lut; memcpy(g.grid_beam, h->grid_beam, sizeof(g.grid_beam)); memcpy(g.grid, h->grid, sizeof(g.grid));
            std::lock_guard<std::mutex> lk(mu);
            cache.push_back(g);
        }
    }
    h->fl = (p.flags == (VPMC_FLAG_MCS | VPMC_FLAG_STRAGGLE | VPMC_FLAG_NUCLEAR)) ? 1 : 0;
#undef CUC
#undef CUA
    *out = h;
    return VPMC_OK;
}

extern "C" const char *vpmc_last_error(const vpmc_t *h) { return h ? h->err.c_str() : g_create_err.c_str(); }

extern "C" int vpmc_add_beam(vpmc_t *h, const vpmc_frame *frame, int *beam_id)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    if (!frame) FAIL(h, VPMC_ERR_INVALID_ARG, "frame is NULL");
    // rot must be orthonormal (1e-3)
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            double d = 0;
            for (int k = 0; k < 3; ++k) d += (double)frame->rot[3 * k + i] * frame->rot[3 * k + j];
            if (std::fabs(d - (i == j ? 1.0 : 0.0)) > 1e-3) FAIL(h, VPMC_ERR_INVALID_ARG, "frame.rot is not orthonormal");
        }
    if (h->beams.size() >= 255) FAIL(h, VPMC_ERR_INVALID_ARG, "at most 255 beams");
    BeamHost b;
    b.frame = *frame;
    h->beams.push_back(b);
    h->spots_dirty = true;
    if (beam_id) *beam_id = (int)h->beams.size() - 1;
    return VPMC_OK;
}

static int check_beam(vpmc_t *h, int beam)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    if (beam < 0 || beam >= (int)h->beams.size()) FAIL(h, VPMC_ERR_INVALID_ARG, "no beam %d", beam);
    return VPMC_OK;
}

extern "C" int vpmc_set_beam(vpmc_t *h, int beam, const vpmc_spot *spots, int32_t n_spots)
{
    int rc = check_beam(h, beam); if (rc) return rc;
    if (n_spots < 0 || (n_spots > 0 && !spots)) FAIL(h, VPMC_ERR_INVALID_ARG, "bad spot list");
    for (int j = 0; j < n_spots; ++j)
        if (!(spots[j].energy > 0) || !(spots[j].weight >= 0) || !(spots[j].sigma >= 0)) FAIL(h, VPMC_ERR_INVALID_ARG, "bad spot %d", j);
    h->beams[beam].spots.assign(spots, spots + n_spots);
    h->spots_dirty = true;
    return VPMC_OK;
}

extern "C" int vpmc_set_range_shifter(vpmc_t *h, int beam, float wet_mm, float downstream_face_mm)
{
    int rc = check_beam(h, beam); if (rc) return rc;
    if (!(wet_mm >= 0)) FAIL(h, VPMC_ERR_INVALID_ARG, "negative WET");
    h->beams[beam].rs_wet = wet_mm;
    h->beams[beam].rs_face = downstream_face_mm > 0 ? downstream_face_mm : 190.0f;
    h->spots_dirty = true;
    return VPMC_OK;
}

extern "C" int vpmc_set_aperture(vpmc_t *h, int beam, float thickness_mm, int material, const uint8_t *opening,
                                 int32_t nx, int32_t ny, float u0, float v0, float du, float dv, float downstream_face_mm)
{
    int rc = check_beam(h, beam); if (rc) return rc;
    BeamHost &b = h->beams[beam];
    if (!(thickness_mm >= 0)) FAIL(h, VPMC_ERR_INVALID_ARG, "negative thickness");
    if (thickness_mm == 0) { free_beam(h, b); b.has_ap = false; h->spots_dirty = true; return VPMC_OK; }
    if (material != VPMC_BRASS) FAIL(h, VPMC_ERR_INVALID_ARG, "only VPMC_BRASS is supported");
    if (!opening || nx < 1 || ny < 1 || nx > 16384 || ny > 16384 || !(du > 0) || !(dv > 0)) FAIL(h, VPMC_ERR_INVALID_ARG, "bad opening bitmap");
    // S0 on the device (vpmc_setup.cuh): bitmap packing and the two safe-distance maps.  Tile = 2^kApTileShift
    // pixels squared; map 0 = Chebyshev distance in tiles to the nearest tile that is not fully open (everything outside the
    // bitmap is brass), map 1 = to the nearest tile that holds any open pixel; both exact, capped at 255.
    const int rw = (nx + 31) / 32;
    const int ts = 1 << kApTileShift, ntx = (nx + ts - 1) / ts, nty = (ny + ts - 1) / ts;
    const size_t npix = (size_t)nx * ny, ntile = (size_t)ntx * nty;
    free_beam(h, b);
    int rc2;
    if ((rc2 = dev_alloc(h, (void **)&b.d_bits, (size_t)rw * ny * sizeof(uint32_t))) || (rc2 = dev_alloc(h, (void **)&b.d_dist, 2 * ntile)) ||
        (rc2 = dev_alloc(h, (void **)&b.d_ap_tmp, npix + 3 * ntile))) return rc2;
    unsigned char *d_open = b.d_ap_tmp, *d_flags = d_open + npix, *d_cbr = d_flags + ntile, *d_cop = d_cbr + ntile;
    cudaStream_t ss = h->setup_stream;
    CU(h, cudaMemcpyAsync(d_open, opening, npix, cudaMemcpyHostToDevice, ss));
    CU(h, cudaEventRecord(h->copy_ev, ss));
    ap_pack_kernel<<<(unsigned)(((size_t)rw * 32 * ny + 255) / 256), 256, 0, ss>>>(d_open, nx, ny, rw, b.d_bits);
    ap_tile_flags_kernel<<<(unsigned)((ntile + 255) / 256), 256, 0, ss>>>(d_open, nx, ny, kApTileShift, ntx, nty, d_flags);
    ap_dist_columns_kernel<<<(ntx + 63) / 64, 64, 0, ss>>>(d_flags, ntx, nty, d_cbr, d_cop);
    ap_dist_rows_kernel<<<(unsigned)((2 * ntile + 255) / 256), 256, 0, ss>>>(d_cbr, d_cop, ntx, nty, b.d_dist);
    CU(h, cudaGetLastError());
    h->launches += 4;
    h->setup_pending = true;
    b.ap_ntx = ntx; b.ap_nty = nty;
    b.has_ap = true; b.ap_T = thickness_mm; b.ap_face = downstream_face_mm > 0 ? downstream_face_mm : 150.0f;
    b.ap_nx = nx; b.ap_ny = ny; b.ap_row_words = rw; b.ap_u0 = u0; b.ap_v0 = v0; b.ap_du = du; b.ap_dv = dv;
    h->spots_dirty = true;
    CU(h, cudaEventSynchronize(h->copy_ev));       // the caller's bitmap is copied during the call
    return VPMC_OK;
}

extern "C" int vpmc_set_aperture_polygon(vpmc_t *h, int beam, float thickness_mm, int material, const float *vertices_xy, int32_t n_vertices,
                                         float downstream_face_mm)
{
    int rc = check_beam(h, beam); if (rc) return rc;
    BeamHost &b = h->beams[beam];
    if (!(thickness_mm > 0)) FAIL(h, VPMC_ERR_INVALID_ARG, "thickness must be positive (use vpmc_set_aperture with 0 to remove the block)");
    if (material != VPMC_BRASS) FAIL(h, VPMC_ERR_INVALID_ARG, "only VPMC_BRASS is supported");
    if (!vertices_xy || n_vertices < 3 || n_vertices > (1 << 20)) FAIL(h, VPMC_ERR_INVALID_ARG, "a polygon needs 3 .. 2^20 vertices");
    float lo[2] = { vertices_xy[0], vertices_xy[1] }, hi[2] = { vertices_xy[0], vertices_xy[1] };
    for (int k = 0; k < n_vertices; ++k)
        for (int a = 0; a < 2; ++a) {
            const float v = vertices_xy[2 * k + a];
            if (!std::isfinite(v)) FAIL(h, VPMC_ERR_INVALID_ARG, "vertex %d is not finite", k);
            lo[a] = std::min(lo[a], v); hi[a] = std::max(hi[a], v);
        }
    const float ext = std::max(hi[0] - lo[0], hi[1] - lo[1]);
    if (!(ext > 0)) FAIL(h, VPMC_ERR_INVALID_ARG, "degenerate polygon");
    // coarse grid: ~96 cells across the larger extent, one cell of margin all round
    const float cell = ext / 96.0f;
    const int nx = (int)std::ceil((hi[0] - lo[0]) / cell) + 2, ny = (int)std::ceil((hi[1] - lo[1]) / cell) + 2;
    // per grid row: the edges whose y-range meets the row, widened by a margin that covers the rounding of the row lookup
    const float x0 = lo[0] - cell, y0 = lo[1] - cell, margin = 1e-3f * cell + 1e-4f;
    std::vector<int> rows((size_t)ny + 1, 0), edges;
    {
        std::vector<std::vector<int>> lists((size_t)ny);
        for (int k = 0; k < n_vertices; ++k) {
            const float ya = vertices_xy[2 * k + 1], yb = vertices_xy[2 * ((k + 1) % n_vertices) + 1];
            const int r0 = std::max((int)std::floor((std::min(ya, yb) - margin - y0) / cell), 0);
            const int r1 = std::min((int)std::floor((std::max(ya, yb) + margin - y0) / cell), ny - 1);
            for (int r = r0; r <= r1; ++r) lists[r].push_back(k);
        }
        for (int r = 0; r < ny; ++r) { rows[r + 1] = rows[r] + (int)lists[r].size(); edges.insert(edges.end(), lists[r].begin(), lists[r].end()); }
    }
    rows.insert(rows.end(), edges.begin(), edges.end());
    free_beam(h, b);
    if ((rc = dev_alloc(h, (void **)&b.d_poly, (size_t)n_vertices * sizeof(float2))) || (rc = dev_alloc(h, (void **)&b.d_pgrid, (size_t)nx * ny * sizeof(float))) ||
        (rc = dev_alloc(h, (void **)&b.d_prows, rows.size() * sizeof(int)))) return rc;
    cudaStream_t ss = h->setup_stream;
    CU(h, cudaMemcpyAsync(b.d_poly, vertices_xy, (size_t)n_vertices * sizeof(float2), cudaMemcpyHostToDevice, ss));
    CU(h, cudaMemcpyAsync(b.d_prows, rows.data(), rows.size() * sizeof(int), cudaMemcpyHostToDevice, ss));
    CU(h, cudaEventRecord(h->copy_ev, ss));
    b.pg_nx = nx; b.pg_ny = ny; b.pg_cell = cell; b.pg_x0 = x0; b.pg_y0 = y0;
    polygon_grid_kernel<<<(nx * ny + 127) / 128, 128, 0, ss>>>(b.d_poly, n_vertices, nx, ny, b.pg_x0, b.pg_y0, cell, b.d_pgrid);
    CU(h, cudaGetLastError());
    h->launches += 1;
    h->setup_pending = true;
    b.ap_n_poly = n_vertices;
    b.has_ap = true; b.ap_T = thickness_mm; b.ap_face = downstream_face_mm > 0 ? downstream_face_mm : 150.0f;
    b.ap_nx = b.ap_ny = 0; b.ap_row_words = 0; b.ap_ntx = b.ap_nty = 0;
    h->spots_dirty = true;
    CU(h, cudaEventSynchronize(h->copy_ev));       // the caller's vertices are copied during the call
    return VPMC_OK;
}

extern "C" int vpmc_get_aperture_tables(vpmc_t *h, int beam, uint32_t *bits_out_host, uint8_t *dist_out_host, int32_t *dims_out)
{
    int rc = check_beam(h, beam); if (rc) return rc;
    const BeamHost &b = h->beams[beam];
    if (!b.has_ap || b.ap_n_poly > 0) FAIL(h, VPMC_ERR_STATE, "beam %d has no bitmap aperture", beam);
    if (dims_out) { dims_out[0] = b.ap_row_words; dims_out[1] = b.ap_ny; dims_out[2] = b.ap_ntx; dims_out[3] = b.ap_nty; }
    CU(h, cudaStreamSynchronize(h->setup_stream));
    if (bits_out_host) CU(h, cudaMemcpy(bits_out_host, b.d_bits, (size_t)b.ap_row_words * b.ap_ny * sizeof(uint32_t), cudaMemcpyDeviceToHost));
    if (dist_out_host) CU(h, cudaMemcpy(dist_out_host, b.d_dist, (size_t)2 * b.ap_ntx * b.ap_nty, cudaMemcpyDeviceToHost));
    return VPMC_OK;
}

static ScoreGeom score_geom(const vpmc_t *h)
{
    ScoreGeom g;
    g.on = h->d_cell_rho ? 1 : 0;
    g.dx = h->sdiv[0]; g.dy = h->sdiv[1]; g.dz = h->sdiv[2]; g.snx = h->sn[0]; g.sny = h->sn[1];
    return g;
}

extern "C" int vpmc_set_scoring_grid(vpmc_t *h, int32_t div_x, int32_t div_y, int32_t div_z)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    if (div_x < 1 || div_y < 1 || div_z < 1 || div_x > h->G.nx || div_y > h->G.ny || div_z > h->G.nz) FAIL(h, VPMC_ERR_INVALID_ARG, "scoring divisors must be in [1, n] per axis");
    dev_release(h, h->d_cell_rho); dev_release(h, h->d_s1); dev_release(h, h->d_s2);       // sized by the scoring grid
    h->d_cell_rho = nullptr; h->d_s1 = nullptr; h->d_s2 = nullptr;
    h->sdiv[0] = div_x; h->sdiv[1] = div_y; h->sdiv[2] = div_z;
    const int n[3] = { h->G.nx, h->G.ny, h->G.nz };
    for (int a = 0; a < 3; ++a) h->sn[a] = (n[a] + h->sdiv[a] - 1) / h->sdiv[a];
    h->ncell = (long long)h->sn[0] * h->sn[1] * h->sn[2];
    h->unc_valid = false;
    if (div_x == 1 && div_y == 1 && div_z == 1) return VPMC_OK;
    int rc = dev_alloc(h, (void **)&h->d_cell_rho, (size_t)h->ncell * sizeof(float)); if (rc) return rc;
    // the per-voxel buffers of the uncertainty estimate keep their (larger) size
    cell_rho_kernel<<<(unsigned)((h->ncell + 127) / 128), 128, 0, h->setup_stream>>>(h->d_hu, h->d_lut, h->G, h->params.rho_min, score_geom(h), h->sn[2], h->d_cell_rho);
    CU(h, cudaGetLastError());
    h->launches += 1;
    h->setup_pending = true;
    return VPMC_OK;
}

extern "C" int vpmc_get_scoring_dims(vpmc_t *h, int32_t *dims_out)
{
    if (!h || !dims_out) return VPMC_ERR_INVALID_ARG;
    for (int a = 0; a < 3; ++a) dims_out[a] = h->sn[a];
    return VPMC_OK;
}

extern "C" int vpmc_set_history_window(vpmc_t *h, uint64_t hid_begin, uint64_t hid_end)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    h->win_lo = hid_begin; h->win_hi = hid_end;
    return VPMC_OK;
}

extern "C" int vpmc_set_shard(vpmc_t *h, int32_t index, int32_t count)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    if (count < 1 || index < 0 || index >= count) FAIL(h, VPMC_ERR_INVALID_ARG, "shard %d of %d", index, count);
    h->shard_index = index; h->shard_count = count;
    return VPMC_OK;
}

// ---- per-kernel-class timing (events on the launching stream) ----
struct TimedScope {
    vpmc_t *h; cudaStream_t st; int cls; cudaEvent_t a = nullptr, b = nullptr;
    TimedScope(vpmc_t *h_, cudaStream_t st_, int cls_, bool enabled = true) : h(h_), st(st_), cls(cls_)
    {
        if (enabled && h->timing && cudaEventCreate(&a) == cudaSuccess && cudaEventCreate(&b) == cudaSuccess) cudaEventRecord(a, st);
        else a = nullptr;
    }
    ~TimedScope()
    {
        if (a) { cudaEventRecord(b, st); h->timed.push_back({ a, b, cls }); }
    }
};

extern "C" int vpmc_set_timing(vpmc_t *h, int on)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    h->timing = on != 0;
    return VPMC_OK;
}

extern "C" int vpmc_get_timing(vpmc_t *h, double *ms_out, uint64_t *launches_out)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    if (!ms_out || !launches_out) FAIL(h, VPMC_ERR_INVALID_ARG, "NULL argument");
    for (int i = 0; i < VPMC_N_KERNEL_CLASSES; ++i) { ms_out[i] = 0.0; launches_out[i] = 0; }
    for (auto &t : h->timed) {
        CU(h, cudaEventSynchronize(t.b));
        float ms = 0.0f;
        CU(h, cudaEventElapsedTime(&ms, t.a, t.b));
        ms_out[t.cls] += ms; launches_out[t.cls] += 1;
        cudaEventDestroy(t.a); cudaEventDestroy(t.b);
    }
    h->timed.clear();
    return VPMC_OK;
}

extern "C" int vpmc_bench_red(vpmc_t *h, uint64_t buffer_bytes, uint64_t n_ops, double *ms_out, uint64_t *n_ops_out)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    if (!ms_out || !n_ops_out || buffer_bytes < 1024 || buffer_bytes > ((uint64_t)1 << 32) || (buffer_bytes & (buffer_bytes - 1)) || n_ops < 1)
        FAIL(h, VPMC_ERR_INVALID_ARG, "bench_red: buffer_bytes must be a power of two in [2^10, 2^32], n_ops >= 1");
    DevBuf buf;
    int rc = ensure(h, buf, (size_t)buffer_bytes); if (rc) return rc;
    const int grid = h->n_sm * 8, block = 256;
    const unsigned long long threads = (unsigned long long)grid * block;
    const unsigned int per = (unsigned int)std::min<unsigned long long>(std::max<unsigned long long>(n_ops / threads, 1ull), 1ull << 24);
    cudaEvent_t a = nullptr, b = nullptr;
    cudaError_t e = cudaMemset(buf.p, 0, (size_t)buffer_bytes);
    if (e == cudaSuccess) e = cudaEventCreate(&a);
    if (e == cudaSuccess) e = cudaEventCreate(&b);
    if (e == cudaSuccess) {
        red_ceiling_kernel<<<grid, block>>>(buf.as<float>(), (unsigned int)(buffer_bytes / 4 - 1), std::min(per, 64u));   // warm-up: the buffer into L2
        cudaEventRecord(a);
        red_ceiling_kernel<<<grid, block>>>(buf.as<float>(), (unsigned int)(buffer_bytes / 4 - 1), per);
        cudaEventRecord(b);
        h->launches += 2;
        e = cudaEventSynchronize(b);
    }
    float ms = 0.0f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, a, b);
    if (a) cudaEventDestroy(a);
    if (b) cudaEventDestroy(b);
    cudaDeviceSynchronize();
    pool_give(buf.p, buf.bytes);
    if (e != cudaSuccess) FAIL(h, VPMC_ERR_CUDA, "bench_red: %s", cudaGetErrorString(e));
    *ms_out = (double)ms; *n_ops_out = (uint64_t)per * threads;
    return VPMC_OK;
}

extern "C" int vpmc_set_knob(vpmc_t *h, int knob, double value)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    switch (knob) {
    case VPMC_KNOB_CHUNK:
        if (!(value >= 1024.0 && value <= 1073741824.0)) FAIL(h, VPMC_ERR_INVALID_ARG, "chunk must be in [2^10, 2^30]");
        h->chunk = (unsigned long long)value; break;
    case VPMC_KNOB_BOX_GROW:
        if (!(value >= 0.0 && value <= 4.0)) FAIL(h, VPMC_ERR_INVALID_ARG, "box growth must be in [0, 4]");
        h->box_grow = (float)value; break;
    case VPMC_KNOB_BOX_PAD:
        if (!(value >= 0.0 && value <= 1024.0)) FAIL(h, VPMC_ERR_INVALID_ARG, "box padding must be in [0, 1024]");
        h->box_pad = (int)value; break;
    case VPMC_KNOB_OVF_CAP:
        if (!(value >= 0.0 && value <= 268435456.0)) FAIL(h, VPMC_ERR_INVALID_ARG, "overflow capacity must be in [0, 2^28]");
        h->ovf_cap = (unsigned int)value; break;
    case VPMC_KNOB_OVF_SORT_CAP:
        if (!(value >= 1.0 && value <= (double)kOvfSortCap)) FAIL(h, VPMC_ERR_INVALID_ARG, "overflow sort capacity must be in [1, %d]", kOvfSortCap);
        h->ovf_sort_cap = (unsigned int)value; break;
    case VPMC_KNOB_LUT_GLOBAL:
        h->smem_lut = (value == 0.0) && h->lut_bytes <= kMaxSmemLut; break;
    case VPMC_KNOB_VERBOSE:
        h->verbose = value != 0.0; break;
    default: FAIL(h, VPMC_ERR_INVALID_ARG, "unknown knob %d", knob);
    }
    return VPMC_OK;
}

extern "C" int vpmc_get_launch_count(vpmc_t *h, uint64_t *out)
{
    if (!h || !out) return VPMC_ERR_INVALID_ARG;
    *out = h->launches;
    return VPMC_OK;
}

#include "vpmc_run.inl"

// ---- the entry point that allocates nothing (include/vpmc.h): vpmc_spmv_grad with its scratch in g_spmv_static_part.
// No cudaMalloc / cudaFree / buffer cache / event creation on this path; the two kernels are the ones vpmc_spmv_grad launches.
extern "C" int vpmc_spmv_grad_static(vpmc_t *h, const vpmc_csr *m, const float *r_dev, float *grad_dev, int accumulate, void *cuda_stream)
{
    if (!h) return VPMC_ERR_INVALID_ARG;
    int rc = check_csr(h, m); if (rc) return rc;
    if ((m->n_rows > 0 && !grad_dev) || (m->nnz > 0 && !r_dev)) FAIL(h, VPMC_ERR_INVALID_ARG, "bad spmv_grad_static arguments");
    if (m->nnz > (int64_t)VPMC_STATIC_MAX_NNZ)
        FAIL(h, VPMC_ERR_INVALID_ARG, "vpmc_spmv_grad_static: %lld entries exceed VPMC_STATIC_MAX_NNZ = %lld (the static scratch holds %d chunks of %d entries); use vpmc_spmv_grad",
             (long long)m->nnz, (long long)VPMC_STATIC_MAX_NNZ, kStaticChunks, kSpmvChunk);
    if (!h->static_scratch) FAIL(h, VPMC_ERR_CUDA, "vpmc_spmv_grad_static: no static scratch on device %d: %s", h->device, h->static_scratch_err.c_str());
    cudaStream_t st = (cudaStream_t)cuda_stream;
    h->last_stream = st; h->launched = true;
    const int nc = spmv_chunks(m->nnz);
    // every partial the fix-up reads is written by the gather of the same call: nothing in the scratch has to start at zero
    float *fp = h->static_scratch, *lp = fp + kStaticChunks;
    if (nc > 0) {
        spmv_grad_kernel<<<nc, kSpmvBlock, 0, st>>>((const long long *)m->row_ptr, m->col, m->val, m->n_rows, m->nnz, r_dev, grad_dev, accumulate, fp, lp);
        h->launches += 1;
    }
    if (m->n_rows > 0) {
        spmv_grad_fixup_kernel<<<(m->n_rows + 255) / 256, 256, 0, st>>>((const long long *)m->row_ptr, m->n_rows, fp, lp, grad_dev, accumulate);
        h->launches += 1;
    }
    CU(h, cudaGetLastError());
    return VPMC_OK;
}
