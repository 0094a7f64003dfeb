// vpmc_host.h -- host-side state of one engine handle (not part of the public ABI).
#pragma once
#include <cuda_runtime.h>

#include <cstdint>
#include <string>
#include <vector>

#include "../../include/vpmc.h"
#include "vpmc_kernels.cuh"

struct BeamHost {
    vpmc_frame frame;
    std::vector<vpmc_spot> spots;
    float rs_wet = 0.0f, rs_face = 190.0f;
    bool has_ap = false;
    float ap_T = 0.0f, ap_face = 150.0f;
    int ap_nx = 0, ap_ny = 0, ap_row_words = 0;
    float ap_u0 = 0, ap_v0 = 0, ap_du = 1, ap_dv = 1;
    uint32_t *d_bits = nullptr;       // packed opening bitmap on the device
};

struct vpmc {
    vpmc_params params;
    vpk::DevParams P;
    vpk::DevGrid G;
    long long nvox = 0;
    int device = 0, n_sm = 0;

    // device-resident inputs
    short *d_hu = nullptr;
    float4 *d_lut = nullptr;          // per-HU (rsp, rho, xsp/X0_w, za_w*rho)
    std::vector<BeamHost> beams;
    bool spots_dirty = true;
    int n_spots = 0;
    float4 *d_spots = nullptr;        // x, y, E, sigma
    double *d_spot_R0 = nullptr;      // alpha E^p per spot, fp64
    int *d_spot_beam = nullptr;
    vpk::DevBeam *d_beams = nullptr;
    std::vector<double> spot_w;       // weights in global spot order
    std::vector<int> spot_beam_h;

    // work mapping
    unsigned long long *d_cum = nullptr, *d_first = nullptr;
    int map_capacity = 0;

    // survivor queue
    vpk::Queue q{};
    unsigned int *d_qctr = nullptr;   // [0] count, [1] head

    // scoring
    float *d_edep = nullptr;          // current batch E_dep (MeV)
    float *d_sum = nullptr, *d_s1 = nullptr, *d_s2 = nullptr;
    vpk::DevTallies *d_tal = nullptr;
    unsigned int *d_max_bits = nullptr;
    double *d_unc = nullptr;          // [0] sum, [1] count
    bool unc_valid = false;

    // influence scratch (grown on demand)
    void *d_inf[16] = { nullptr };
    size_t inf_bytes[16] = { 0 };

    // launch configuration
    int voxel_grid[2][2] = { { 0, 0 }, { 0, 0 } };   // [mode][smem_lut]
    bool smem_lut = false;
    size_t lut_bytes = 0;

    unsigned long long win_lo = 0, win_hi = 0;
    cudaStream_t last_stream = nullptr;
    unsigned long long launches = 0;
    bool timing = false;
    struct Timed { cudaEvent_t a, b; int cls; };
    std::vector<Timed> timed;
    std::string err;
};
