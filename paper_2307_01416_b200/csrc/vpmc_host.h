// vpmc_host.h -- host-side state of one engine handle (not part of the public ABI).
#pragma once
#include <cuda_runtime.h>

#include <cstdint>
#include <string>
#include <vector>

#include "../../include/vpmc.h"
#include "vpmc_kernels.cuh"
#include "vpmc_spmv.cuh"
#include "vpmc_gamma.cuh"

struct BeamHost {
    vpmc_frame frame;
    std::vector<vpmc_spot> spots;
    float rs_wet = 0.0f, rs_face = 190.0f;
    bool has_ap = false;
    float ap_T = 0.0f, ap_face = 150.0f;
    int ap_nx = 0, ap_ny = 0, ap_row_words = 0;
    float ap_u0 = 0, ap_v0 = 0, ap_du = 1, ap_dv = 1;
    uint32_t *d_bits = nullptr;       // packed opening bitmap on the device
    unsigned char *d_dist = nullptr;  // safe-distance maps of the opening, one byte per tile of 2^kApTileShift pixels: to brass, then to the opening
    unsigned char *d_ap_tmp = nullptr;    // set-up scratch: the caller's uint8 bitmap, tile flags, column distances
    int ap_ntx = 0, ap_nty = 0;
    // polygon opening (vpmc_set_aperture_polygon)
    int ap_n_poly = 0;
    float2 *d_poly = nullptr;
    float *d_pgrid = nullptr;
    int *d_prows = nullptr;           // row_ptr [pg_ny + 1] followed by the edge lists
    int pg_nx = 0, pg_ny = 0;
    float pg_x0 = 0, pg_y0 = 0, pg_cell = 1;
};

// a device buffer that only grows
struct DevBuf {
    void *p = nullptr;
    size_t bytes = 0;
    template <class T> T *as() const { return static_cast<T *>(p); }
};

struct vpmc {
    vpmc_params params;
    vpk::DevParams P;
    vpk::DevGrid G;
    long long nvox = 0;
    int device = 0, n_sm = 0;
    // scoring grid (S:8f-4, vpmc_set_scoring_grid): cells of sdiv voxels per axis; ncell = nvox and d_cell_rho = NULL by default
    int sdiv[3] = { 1, 1, 1 }, sn[3] = { 0, 0, 0 };
    long long ncell = 0;
    float *d_cell_rho = nullptr;      // per cell: sum over its voxels of max(rho, rho_min)

    // Device memory of the fixed-size members below comes from the process-wide buffer cache (vpmc_api.cu) and goes back to
    // it in vpmc_destroy.  Set-up work (uploads, S0 kernels) is enqueued on setup_stream; the next compute call makes its
    // stream wait for it.
    struct Owned { void *p; size_t bytes; };
    std::vector<Owned> owned;
    cudaStream_t setup_stream = nullptr;
    cudaEvent_t setup_ev = nullptr, copy_ev = nullptr;
    bool setup_pending = false;
    bool launched = false;            // some compute call has enqueued work on last_stream

    // device-resident inputs
    short *d_hu = nullptr;
    float4 *d_lut = nullptr;          // per-HU (rsp, rho, xsp/X0_w, 1/rsp)
    std::vector<BeamHost> beams;
    bool spots_dirty = true;
    int n_spots = 0;
    float4 *d_spots = nullptr;        // x, y, E, sigma
    double *d_spot_R0 = nullptr;      // alpha E^p per spot, fp64
    int *d_spot_beam = nullptr;
    vpk::DevBeam *d_beams = nullptr;
    std::vector<double> spot_w;       // weights in global spot order
    std::vector<int> spot_beam_h;

    // work mapping (dose mode): [n_batches * n_spots + 1]
    DevBuf cum, first;
    DevBuf s0, s1, s2;                // range-shifter records of a chunk
    DevBuf a0, a1, a2, a3, a4;        // queue range shifter -> aperture entry
    DevBuf b0, b1, b2, b3, b4, b5;    // aperture queue (histories whose next step is a brass step)
    DevBuf q0, q1, q2, q3, q4;        // CT queue (all grown to the chunk size in use)
    unsigned int *d_qctr = nullptr;   // counts and heads of the queues of the chunk in flight (vpmc_run.inl)
    bool any_rs = false, any_ap = false;

    // scoring
    DevBuf edep;                      // [n_batches][nvox] E_dep (MeV)
    float *d_s1 = nullptr, *d_s2 = nullptr, *d_fb = nullptr;
    vpk::DevTallies *d_tal = nullptr, *d_tal_scratch = nullptr;
    unsigned int *d_max_bits = nullptr;
    double *d_unc = nullptr;          // [0] sum, [1] count
    bool unc_valid = false;

    // sequential stopping rule (vpmc_dose_to_uncertainty)
    vpk::SeqState *d_seq = nullptr;
    cudaStream_t seq_stream = nullptr;    // capture needs a non-default stream
    cudaEvent_t seq_ev_in = nullptr, seq_ev_out = nullptr;
    cudaGraph_t seq_graph = nullptr;
    cudaGraphExec_t seq_exec = nullptr;
    bool seq_valid = false;

    // influence workspace (grown on demand)
    DevBuf inf_scratch, inf_lo, inf_dim, inf_off, inf_bbox, inf_cols, inf_tile0, inf_tilecol, inf_skip, inf_tilecnt, inf_colmax,
        inf_colnnz, inf_colbase, inf_stage_idx, inf_stage_val, inf_rowsrc,
        ovf_key, ovf_val, ovf_key2, ovf_val2, ovf_flag, ovf_colcnt, ovf_coloff, ovf_kept, ovf_ctr, ostage_idx, ostage_val, row_ovf_off, row_ovf_n;
    vpmc_influence_stats inf_stats = {};
    DevBuf gamma_buf;                 // counters + list of the voxels that fail the zero-distance test (vpmc_gamma)
    DevBuf spmv_part;                 // first / last partial sums per chunk of vpmc_spmv_grad
    float *static_scratch = nullptr;  // device address of the file-scope scratch of vpmc_spmv_grad_static on h->device (vpmc_api.cu)
    std::string static_scratch_err;
    size_t workspace_limit = 0;       // bytes of influence scratch per group (0 = automatic)

    // knobs (vpmc_set_knob)
    unsigned long long chunk = 1ull << 23;   // work items per pass of the pipeline = queue capacity
    float box_grow = 0.05f;           // influence: growth of the pilot box, fraction of its extent
    int box_pad = 1;                  // influence: extra voxels per side
    unsigned int ovf_cap = 1u << 25;  // influence: entries of the overflow list (12 B each)
    unsigned int ovf_sort_cap = vpk::kOvfSortCap;   // influence: overflow entries of one column beyond which the column is replayed
    bool verbose = false;

    // launch configuration
    // resident CTAs of beam_kernel<STAGE, FL> [stage][fl] and voxel_kernel<MODE, SMEM_LUT, FL> [mode][smem_lut][fl]; fl = 1: the
    // kernels specialised for the default physics switches (flags == 7), 0: the switches read at run time
    int grid_beam[2][2] = {};
    int grid[3][2][2] = {};
    int fl = 1;
    bool smem_lut = false;
    size_t lut_bytes = 0, tally_smem = 0;

    unsigned long long win_lo = 0, win_hi = 0;
    int shard_index = 0, shard_count = 1;     // vpmc_set_shard (S:8e)
    cudaStream_t last_stream = nullptr;
    unsigned long long launches = 0;
    bool timing = false;
    struct Timed { cudaEvent_t a, b; int cls; };
    std::vector<Timed> timed;
    std::string err;
};
