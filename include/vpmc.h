/*
 * vpmc.h -- C-ABI of libvpmc.so: B200-native (sm_100a) Monte Carlo proton transport-and-scoring loop of
 * arXiv 2307.01416 ("block aperture in VPMC"): spot source -> range shifter -> brass aperture -> voxelised
 * CT -> dose grid / per-spot sparse influence columns.
 *
 * Citations: P:Lnn = PAPER.md line nn; S:8x = SURVEY.md section 8(x) (the written-out closed-form reading
 * of what the paper defers to its ref. 65); D:Rn = DESIGN.md reading n.
 *
 * General conventions
 *   - Units: mm, MeV, radians; dose in Gy per unit spot weight (weights are proton counts).
 *   - Every call returns VPMC_OK (0) or a negative VPMC_ERR_*; nothing throws or aborts across the ABI.
 *     vpmc_last_error() gives a message for the last failing call on that handle (or on create, with NULL).
 *   - Pointers marked [host] are caller-owned host memory, copied during the call.  Pointers marked
 *     [device] are caller-owned CUDA device memory on the current device.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = default stream).  Work is enqueued on it.
 *   - Same handle + same seed + same inputs => identical integer outputs; floating-point sums equal up
 *     to the order of atomic additions.
 *   - There is no CPU fallback: without a CUDA device every compute call returns VPMC_ERR_CUDA.
 */
#ifndef VPMC_H_
#define VPMC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define VPMC_OK 0
#define VPMC_ERR_INVALID_ARG (-1)
#define VPMC_ERR_GEOMETRY (-2)   /* e.g. CT box overlaps the aperture, range shifter not upstream of aperture */
#define VPMC_ERR_CUDA (-3)
#define VPMC_ERR_ALLOC (-4)
#define VPMC_ERR_STATE (-5)      /* e.g. dose before any beam was set */

#define VPMC_FLAG_MCS 1
#define VPMC_FLAG_STRAGGLE 2
#define VPMC_FLAG_NUCLEAR 4

#define VPMC_BRASS 1             /* aperture material; the only one */

/* step-record codes (vpmc_trace) */
#define VPMC_REG_VACUUM 0
#define VPMC_REG_RS 1
#define VPMC_REG_AP_OPEN 2
#define VPMC_REG_AP_BRASS 3
#define VPMC_REG_CT 4
#define VPMC_CAUSE_CONT 0
#define VPMC_CAUSE_STOPPED 1
#define VPMC_CAUSE_NUCLEAR 2
#define VPMC_CAUSE_ESCAPED 3

typedef struct vpmc vpmc_t;      /* opaque, owned by the library */

/* S:8c-C0.  Physics and stepping parameters; vpmc_default_params() fills the defaults listed there. */
typedef struct {
    float alpha, p;              /* Bragg-Kleeman range in water R = alpha E^p: 0.022 mm MeV^-p, 1.77 */
    float X0_w;                  /* radiation length of water, 360.8 mm */
    float Es, c_log;             /* Highland constants 13.6 MeV, 0.038 */
    float beta_nuc, gamma_loc;   /* nuclear slope 0.0012 /mm of residual range; locally absorbed fraction 0.6 */
    float k_bohr, za_w;          /* Bohr variance 0.015692 MeV^2/mm per (Z/A rho); Z/A of water 0.5551 */
    float R_cut, f_R, s_max;     /* stop at residual range 0.1 mm; step <= max(f_R R, R_cut) WET; geometric cap (inf) */
    float s_rs, s_ap;            /* fixed geometric step in range shifter / aperture region, 1 mm */
    float brass_rsp, brass_rho, brass_X0, brass_za; /* 5.523, 8.5 g/cm3, 14.94 mm, 0.457 */
    float rs_rsp, rs_rho, rs_X0; /* range shifter as water-equivalent slab: 1, 1, 360.8 mm */
    float rho_min;               /* density floor in the dose conversion, 1e-3 g/cm3 */
    float delta_E;               /* relative source energy spread, 0 */
    int32_t flags;               /* VPMC_FLAG_* ; default all three */
    int32_t n_batches;           /* batches of the uncertainty estimate (S:8c-C6, D:R7); default 10; 1 = off */
} vpmc_params;

/* CT grid.  Voxel v = ix + nx*(iy + ny*iz); `origin` is the low corner of voxel (0,0,0) in the CT
 * frame.  hu: nx*ny*nz int16, [host] or, when hu_on_device != 0, [device]. */
typedef struct {
    int32_t n[3];
    float h[3];
    float origin[3];
    const int16_t *hu;
    int32_t hu_on_device;
} vpmc_ct;

/* HU -> (RSP, density g/cm3, relative scattering power) calibration: piecewise linear between nodes
 * ascending in hu, clamped at the end nodes (S:8c-C5).  xsp may be NULL -> rho.  All [host]. */
typedef struct {
    int32_t n;
    const float *hu, *rsp, *rho, *xsp;
} vpmc_calib;

/* One pencil-beam spot: position at the isocentre plane in the beam frame, energy,
 * weight (proton count), in-air Gaussian sigma. */
typedef struct { float x, y, energy, weight, sigma; } vpmc_spot;

/* Beam frame -> CT frame: r_ct = iso + rot * r_beam (rot row-major, orthonormal); the beam travels along
 * +w (third beam axis); the isocentre is w = 0. */
typedef struct { float iso[3]; float rot[9]; } vpmc_frame;

/* Uncertainty scenario: patient shift (mm, CT frame; devices ride on the nozzle) and RSP scale. */
typedef struct { float shift[3]; float rsp_scale; } vpmc_scenario;

/* One scenario's influence matrix in CSR form ("sparse matrix compression"): rows = spots in input
 * order over all beams, columns = voxel linear index ascending.  Arrays are [device], obtained through the
 * caller's allocator and caller-owned afterwards. */
typedef struct {
    int64_t *row_ptr;            /* n_rows + 1 */
    int32_t *col;                /* nnz */
    float *val;                  /* nnz, Gy per unit spot weight */
    int64_t nnz;
    int32_t n_rows;
} vpmc_csr;

/* Allocator callback: must return device memory of at least `bytes` bytes (256-byte aligned), or NULL. */
typedef void *(*vpmc_alloc_fn)(size_t bytes, void *user);

/* Energy bookkeeping (S:8c-P6): incident = dep_ct + dep_rs + dep_brass + escaped + removed. */
typedef struct {
    double incident, dep_ct, dep_rs, dep_brass, escaped, removed;                   /* MeV */
    uint64_t n_stopped_ct, n_stopped_rs, n_stopped_brass, n_nuclear, n_escaped;     /* histories by fate */
    uint64_t n_steps_ct, n_steps_dev;   /* steps taken in the CT / in the beam line (drifts included) */
    uint64_t n_steps_slab;              /* material steps among n_steps_dev (range shifter + brass) */
} vpmc_tallies;

/* One step of one history (vpmc_trace).  r, u after the step: beam frame in the beam line, CT frame from the
 * CT-entry drift on.  ivox = voxel at the start of a CT step, else -1. */
typedef struct {
    uint64_t hid;
    int32_t step, region, cause;
    int32_t ivox[3];
    float r[3], u[3];
    float E_before, E_after, s;
    float dep;                   /* energy deposited in the step's cell (CT voxel, range-shifter or brass tally), MeV */
    int32_t pad_;
} vpmc_step_rec;

void vpmc_default_params(vpmc_params *p);

/* Create an engine for one CT + calibration.  Builds the per-HU material table on the
 * device and uploads the CT.  params NULL = defaults.  *out is NULL on failure. */
int vpmc_create(vpmc_t **out, const vpmc_ct *ct, const vpmc_calib *cal, const vpmc_params *params);
int vpmc_destroy(vpmc_t *h);

/* Add a treatment field; returns its index in *beam_id.  Beams keep their order; spot rows of the influence
 * matrices follow beam order then spot order. */
int vpmc_add_beam(vpmc_t *h, const vpmc_frame *frame, int *beam_id);

/* Spots, energies, weights and spot sigmas of a beam.  spots: [host], n_spots >= 0. */
int vpmc_set_beam(vpmc_t *h, int beam, const vpmc_spot *spots, int32_t n_spots);

/* Range shifter: homogeneous slab of water-equivalent thickness wet_mm (0 = none) whose
 * downstream face is downstream_face_mm upstream of the isocentre (<= 0 -> default 190). */
int vpmc_set_range_shifter(vpmc_t *h, int beam, float wet_mm, float downstream_face_mm);

/* Aperture block: brass of thickness_mm (0 = none) with a patient-specific opening given as a
 * bitmap, opening[iy*nx + ix] != 0 = open, pixel (ix, iy) covering [u0 + ix du, u0 + (ix+1) du) x
 * [v0 + iy dv, ...) in the beam frame; everything outside the bitmap is brass.  The downstream face is
 * downstream_face_mm upstream of the isocentre (<= 0 -> default 150).  opening: [host]. */
int vpmc_set_aperture(vpmc_t *h, int beam, float thickness_mm, int material, const uint8_t *opening,
                      int32_t nx, int32_t ny, float u0, float v0, float du, float dv, float downstream_face_mm);

/* Plan dose: n_histories apportioned to the spots by weight (largest remainder, S:8c-C2), transported
 * and scored; dose_out_dev ([device], nx*ny*nz floats) is fully overwritten with
 * dose[v] = (W/N) E_dep[v] / (max(rho_v, rho_min) V_vox) * 1.602176634e-10 Gy (S:8c-C6).
 * Asynchronous on `cuda_stream` except for the small host-side apportionment; tallies and the uncertainty
 * of this run are available through vpmc_get_tallies / vpmc_get_uncertainty (which synchronise). */
int vpmc_dose(vpmc_t *h, uint64_t n_histories, uint64_t seed, float *dose_out_dev, void *cuda_stream);

/* Same under one uncertainty scenario (vpmc_dose = shift 0, rsp_scale 1). */
int vpmc_dose_scenario(vpmc_t *h, const vpmc_scenario *sc, uint64_t n_histories, uint64_t seed,
                       float *dose_out_dev, void *cuda_stream);

/* vpmc_dose with the result copied to dose_out_host ([host], nx*ny*nz floats); synchronous. */
int vpmc_dose_host(vpmc_t *h, uint64_t n_histories, uint64_t seed, float *dose_out_host);

/* Dose to a statistical uncertainty with the stopping rule ON THE DEVICE (S:8d metric 2, S:8f-3; "<0.5 %").
 * Batches of batch_histories histories are transported one after another; batch k (0, 1, ...) is the batch_histories-history
 * plan sample whose history ids are k 2^32 + i (D:R15).  After each batch the C6 estimator over the batches so far (mean over
 * voxels >= 50 % of the maximum of sigma_v / D_v) is evaluated by a kernel, and a CUDA-graph WHILE node repeats the batch
 * pass until at least max(min_batches, 2) batches ran and the estimate <= target_rel_unc, or max_batches ran: no host round
 * trip between batches.  dose_out_dev is the dose of all batches run (C6 with N = batches x batch_histories).
 * batch_histories <= the chunk size (2^23).  Asynchronous on `cuda_stream`; vpmc_get_run_info synchronises. */
int vpmc_dose_to_uncertainty(vpmc_t *h, const vpmc_scenario *sc, uint64_t batch_histories, int32_t min_batches,
                             int32_t max_batches, float target_rel_unc, uint64_t seed, float *dose_out_dev, void *cuda_stream);
/* Result of the last vpmc_dose_to_uncertainty: batches run, the estimate after the last one, whether the target stopped it. */
int vpmc_get_run_info(vpmc_t *h, int32_t *batches_out, float *rel_unc_out, int32_t *reached_target_out);

/* S:8f-2: aperture block whose opening is given as its boundary polygon, as the paper describes it (the medium is
 * decided at every MC step by the crossing-number test of the proton's lateral position against the opening's polygon,
 * ref. 67; P:L61 on why a voxelised opening is too coarse for small apertures).  vertices_xy: [host], n_vertices pairs
 * (x, y) in the beam frame, mm; edge k joins vertex k to vertex k + 1, the last to the first; either orientation; a point is
 * in the opening iff a ray towards +x crosses an odd number of edges.  Everything outside the polygon is brass.  Replaces
 * any opening set before on this beam.  The test runs on the device for every aperture step (tests whose answer is known
 * from the distance to the nearest edge are skipped, D:5.2). */
int vpmc_set_aperture_polygon(vpmc_t *h, int beam, float thickness_mm, int material, const float *vertices_xy, int32_t n_vertices,
                              float downstream_face_mm);

/* Test-only: the device tables S0 builds from an opening bitmap (D:5.2).  dims_out[4] = {words per row, rows, tiles in u,
 * tiles in v}; bits_out_host: rows x words packed bitmap (bit ix & 31 of word ix >> 5); dist_out_host: 2 maps of tiles_v x
 * tiles_u bytes -- Chebyshev distance in tiles (capped at 255) to the nearest tile that is not fully open, with everything
 * outside the bitmap brass, then to the nearest tile holding any open pixel.  Any output pointer may be NULL. */
int vpmc_get_aperture_tables(vpmc_t *h, int beam, uint32_t *bits_out_host, uint8_t *dist_out_host, int32_t *dims_out);

/* S:8f-4, coarse-grid scoring ("memory usage was further reduced by using dynamic voxel spacing"): score on a grid whose
 * cells are div_x x div_y x div_z CT voxels (the last cell of an axis may be smaller); transport is unchanged.  Afterwards
 * every dose grid this handle takes or returns (vpmc_dose*, vpmc_dose_to_uncertainty, vpmc_gamma) has sn_x*sn_y*sn_z elements,
 * sn = ceil(n / div) (vpmc_get_scoring_dims), cell c = cx + sn_x (cy + sn_y cz), and the influence matrices' columns are cells.
 * Dose of a cell = its energy / its mass: (W/N) E_dep[c] / (V_vox sum_{v in c} max(rho_v, rho_min)) x 1.602176634e-10 Gy,
 * which is C6 for (1, 1, 1), the default.  One factor for the whole grid; spacing per organ would need contours (not built). */
int vpmc_set_scoring_grid(vpmc_t *h, int32_t div_x, int32_t div_y, int32_t div_z);
int vpmc_get_scoring_dims(vpmc_t *h, int32_t *dims_out /* [3] */);

/* Restrict the next dose / trace calls to history ids [hid_begin, hid_end) of the N-history run (prefix
 * parity, S:8d).  hid_end = 0 -> no restriction. */
int vpmc_set_history_window(vpmc_t *h, uint64_t hid_begin, uint64_t hid_end);

/* Multi-GPU sharding (S:8e): this handle computes shard `index` of `count` of the following dose / influence calls.
 * Dose: of every (spot, batch) id range [a, b) of the N-history run only the ids [a + (b - a) index / count,
 * a + (b - a)(index + 1) / count) are transported, with the scale W / N of the full run, so the SUM of the dose grids of
 * the `count` shards is the dose of the full run (same history ids, same random streams; equal up to the order of
 * floating-point additions) and every shard holds the same mix of spots.  Influence: only the rows (spots) g with
 * n_spots index / count <= g < n_spots (index + 1) / count are computed; the other rows of the returned CSR are empty, so
 * the full matrix is the concatenation of the shards' entries, row_ptr offset by the exclusive sum of the shards' nnz.
 * No exchange happens inside the library.  (0, 1) = everything (default). */
int vpmc_set_shard(vpmc_t *h, int32_t index, int32_t count);

/* Influence matrices: for each of n_sc scenarios and each spot j (history ids
 * j*hist_per_spot + i), the dose column per unit weight, entries >= rel_threshold * column max (and > 0) kept,
 * written as CSR into out[0..n_sc) through `alloc` (three calls per scenario: row_ptr, col, val).  Synchronises
 * where it must size outputs.  Tallies afterwards cover every history of every scenario once (the pilot and replay
 * passes that only size the per-column boxes are not counted).  On error out[] may be partially filled. */
int vpmc_influence(vpmc_t *h, const vpmc_scenario *sc, int32_t n_sc, uint32_t hist_per_spot,
                   float rel_threshold, uint64_t seed, vpmc_csr *out, vpmc_alloc_fn alloc, void *user,
                   void *cuda_stream);

/* Counts of the last vpmc_influence call (bench.py's writer roofline, S:8d): elements of the per-column boxes that were
 * zeroed and scanned (all groups, scenarios and replays), deposits that went to the overflow list and how many of its
 * entries were kept, columns replayed, groups run. */
typedef struct {
    uint64_t box_elements, ovf_deposits, ovf_kept, columns_replayed, groups, nnz;
} vpmc_influence_stats;
int vpmc_get_influence_stats(vpmc_t *h, vpmc_influence_stats *out);

/* The CSR writer alone (S:8a-S8, D:R10): one row from a dense fp32 column [device] of n voxels.  With
 * col_out/val_out NULL only counts.  *nnz_out [host].  Synchronous. */
int vpmc_csr_from_dense(vpmc_t *h, const float *col_dev, int64_t n, float rel_threshold,
                        int32_t *col_out_dev, float *val_out_dev, int64_t *nnz_out);

/* ---- S:8f-1: one iteration of the robust optimiser on the influence matrices ("0.1-0.3 s per iteration", P:L160
 * "13 uncertainty scenarios were included in the robust optimization").  The paper prints no objective; D:R16 takes
 * the voxel-wise worst case over the scenarios of a weighted quadratic deviation.  A matrix is a vpmc_csr as vpmc_influence
 * returns it (rows = spots, columns = voxels, [device]); vectors are fp32 [device]; everything is enqueued on cuda_stream.
 *
 * vpmc_spmv_dose:  dose[v] = sum_j D[j][v] w[j], v < n_cols; dose_dev (n_cols floats) is overwritten.  fp32 sums by
 *                  atomic additions: equal up to their order.
 * vpmc_spmv_grad:  grad[j] (+)= sum_v D[j][v] r[v] (accumulate != 0 adds to grad_dev); sums in a fixed order: bit-reproducible.
 * vpmc_worst_case: doses_dev, resid_dev: [n_sc][n] row-major.  Per voxel v: e_s = d_s[v] - target[v], s* = the scenario with
 *                  the largest e_s^2 (products rounded to fp32; the lowest index among equals), resid[s*][v] = 2 weight[v]
 *                  e_s*, resid[s][v] = 0 otherwise; *objective_dev (one double, [device]) = sum_v weight[v] e_s*^2.
 * vpmc_robust_iteration: all of it -- n_sc dose products into doses_ws_dev ([n_sc][n_cols]), the worst case into resid_ws_dev
 *                  (same shape) and *objective_dev, then grad_dev[j] = sum_s sum_v D_s[j][v] resid_s[v], scenarios added in
 *                  order.  All matrices must have the same number of rows. */
int vpmc_spmv_dose(vpmc_t *h, const vpmc_csr *m, int64_t n_cols, const float *w_dev, float *dose_dev, void *cuda_stream);
int vpmc_spmv_grad(vpmc_t *h, const vpmc_csr *m, const float *r_dev, float *grad_dev, int accumulate, void *cuda_stream);
int vpmc_worst_case(vpmc_t *h, const float *doses_dev, int32_t n_sc, int64_t n, const float *target_dev, const float *weight_dev,
                    float *resid_dev, double *objective_dev, void *cuda_stream);
int vpmc_robust_iteration(vpmc_t *h, const vpmc_csr *mats, int32_t n_sc, int64_t n_cols, const float *w_dev, const float *target_dev,
                          const float *weight_dev, float *doses_ws_dev, float *resid_ws_dev, float *grad_dev, double *objective_dev,
                          void *cuda_stream);

/* The one entry point that allocates nothing -- for callers that cannot call cudaMalloc (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid it).  vpmc_spmv_grad_static computes exactly what vpmc_spmv_grad computes, with the same
 * two kernels in the same order (bit-identical result), but its scratch -- two partial sums per chunk of 8192 entries -- is a
 * file-scope device array of the library instead of a buffer from the cache: no cudaMalloc, cudaFree, event creation or other
 * allocating call happens inside it, under any input.  The array holds VPMC_STATIC_MAX_NNZ entries' worth of chunks = 256 KB,
 * and every GPU that loads the library keeps those 256 KB until the process exits.  Its device address is looked up once per
 * device in vpmc_create (cudaGetSymbolAddress, with the handle's device current); if that failed, this call returns
 * VPMC_ERR_CUDA with the reason.  m->nnz > VPMC_STATIC_MAX_NNZ is rejected with VPMC_ERR_INVALID_ARG (use vpmc_spmv_grad).
 * ALL calls on a device share the one array, from any handle and any stream: calls that overlap on the GPU race on it and give
 * wrong sums -- enqueue them on one stream, or order them with events.  The array keeps the last call's contents; nothing in
 * it has to start at zero (every partial sum that is read is written earlier in the same call), so nothing is cleared.
 * m, r_dev, grad_dev as for vpmc_spmv_grad, all [device], caller-owned.  Not covered by vpmc_get_timing. */
#define VPMC_STATIC_MAX_NNZ (1LL << 28)
int vpmc_spmv_grad_static(vpmc_t *h, const vpmc_csr *m, const float *r_dev, float *grad_dev, int accumulate, void *cuda_stream);

/* S:8f-3: 3-D gamma index of two dose grids on this engine's CT grid ("3D Gamma passing rate", Table 2; ref. 80),
 * computed on the device.  S:8c-C6: global normalisation -- dose criterion dd_rel x max(ref); voxels with ref >= threshold_rel
 * x max(ref) are evaluated; a voxel passes if |eval - ref| <= criterion at zero distance, else if min over the lattice points
 * of spacing h / sub within dta_mm of (distance / dta)^2 + ((eval interpolated trilinearly, edge values beyond the grid) - ref)^2
 * / criterion^2 is <= 1.  ref_dev, eval_dev: [device] nx*ny*nz floats.  *n_eval_out, *n_fail_out [host]: voxels evaluated, voxels
 * failing; pass rate = 1 - n_fail / n_eval.  Synchronises cuda_stream. */
int vpmc_gamma(vpmc_t *h, const float *ref_dev, const float *eval_dev, float dd_rel, float dta_mm, float threshold_rel, int32_t sub,
               uint64_t *n_eval_out, uint64_t *n_fail_out, void *cuda_stream);

/* Upper bound in bytes on the per-group scratch of vpmc_influence (the dense per-column boxes of one group of spots);
 * 0 = automatic (a third of the free device memory, at most 24 GiB).  Smaller limits only mean more groups. */
int vpmc_set_workspace_limit(vpmc_t *h, uint64_t bytes);

/* Tallies of the last dose / influence call (synchronises the stream it ran on). */
int vpmc_get_tallies(vpmc_t *h, vpmc_tallies *out);

/* Statistical uncertainty of the last vpmc_dose* call (S:8c-C6): mean over voxels with dose >= 50% of the
 * maximum of sigma_v / D_v from n_batches batches.  Needs params.n_batches >= 2. */
int vpmc_get_uncertainty(vpmc_t *h, float *rel_unc_out);

/* Test-only: step records of selected histories.  mode 0 = dose mode with N = n_or_hps; 1 = influence mode
 * with hist_per_spot = n_or_hps.  out_host: n*max_steps records; nrec_host[i] = records of history i. */
int vpmc_trace(vpmc_t *h, const vpmc_scenario *sc, int32_t mode, uint64_t n_or_hps, uint64_t seed,
               const uint64_t *hids, int32_t n, int32_t max_steps, vpmc_step_rec *out_host, int32_t *nrec_host);

/* Test-only: ONE step of the path from a supplied pre-step state (north_star: "histories must agree step-for-step";
 * S:8c-A9).  The tests feed the oracle's pre-step state of every step, so the comparison carries no accumulated
 * difference.  kind selects the step function: the S1 sampler, a vacuum drift to the next device, one range-shifter /
 * aperture-region step (S2 / S3: the medium of an aperture step is decided by the kernel's own bitmap test), the CT
 * entry (C3), or one voxel step (S4 + S5).  r, u: beam frame (r[2] = w) for kinds 0-5, CT frame for kind 6. */
#define VPMC_STEP_SOURCE 0       /* in: hid, spot (global index); out: r, E, tau_star */
#define VPMC_STEP_DRIFT_TO_RS 1
#define VPMC_STEP_RS 2
#define VPMC_STEP_DRIFT_TO_AP 3
#define VPMC_STEP_AP 4
#define VPMC_STEP_CT_ENTRY 5     /* out: r, u in the CT frame, ivox_after = entry voxel */
#define VPMC_STEP_CT 6           /* in: ivox = current voxel */
typedef struct {
    uint64_t hid;
    int32_t kind, step, beam, spot;
    int32_t ivox[3];
    int32_t pad_;
    double r[3], u[3];
    double E, t_rad, tau, tau_star;
} vpmc_state;
typedef struct {
    int32_t region, cause, step_after, n_steps;   /* n_steps > 1: the kernel took several opening drifts at once (D:R14); the
                                                     FIRST is reported */
    int32_t ivox_after[3];
    int32_t pad_;
    double r[3], u[3];           /* after the step, summed from the kernel's own representation (hi + lo, voxel + offset) */
    double E, R, s, dep, t_rad, tau, tau_star;     /* R = residual range carried by the kernel (fp64) */
} vpmc_state_out;
/* states, out: [host], n entries.  Scenario NULL = nominal.  Synchronous.  Needs beams and spots to be set. */
int vpmc_step_from_state(vpmc_t *h, const vpmc_scenario *sc, uint64_t seed, const vpmc_state *states, int32_t n,
                         vpmc_state_out *out);

/* Test-only: one digest per history of the contiguous ids [hid_begin, hid_begin + n) of the N-history dose run: number
 * of step records, FNV-1a hash (offset 14695981039346656037, prime 1099511628211, one round per 32-bit word) over
 * (region, cause, ivox[0..2]) of every record in order, position after the last record, energy left after it, and
 * the energy deposited in the CT.  Lets a test find, among 10^6 histories, the few whose discrete trace or end point
 * differs from the oracle's.  out_host: n entries.  Synchronous. */
typedef struct {
    uint64_t hid, hash;
    int32_t n_rec, cause;
    float r[3];
    float E_last, dep_ct;
    int32_t pad_;
} vpmc_digest;
int vpmc_digests(vpmc_t *h, const vpmc_scenario *sc, uint64_t n_histories, uint64_t seed, uint64_t hid_begin, int32_t n,
                 vpmc_digest *out_host);

/* Test / tuning knobs of one handle (none changes a result beyond the order of floating-point sums; the tests use them
 * to force the rarely taken code paths).  Returns VPMC_ERR_INVALID_ARG for an unknown knob or a value out of range. */
#define VPMC_KNOB_CHUNK 0        /* work items per pass of the pipeline (default 2^23) */
#define VPMC_KNOB_BOX_GROW 1     /* influence: growth of the pilot box, fraction of its extent (default 0.05) */
#define VPMC_KNOB_BOX_PAD 2      /* influence: extra voxels per side (default 1) */
#define VPMC_KNOB_OVF_CAP 3      /* influence: capacity of the overflow list (default 2^25; 0 forces the replay path) */
#define VPMC_KNOB_LUT_GLOBAL 4   /* 1 = never stage the material table in shared memory */
#define VPMC_KNOB_VERBOSE 5      /* 1 = progress lines of the influence path on stderr */
#define VPMC_KNOB_OVF_SORT_CAP 6 /* influence: overflow entries of ONE column a CTA sorts (default and maximum 16384); a column with more
                                    is replayed with a larger box */
int vpmc_set_knob(vpmc_t *h, int knob, double value);

/* Per-kernel-class device timing (bench.py's roofline): when on, every launch is bracketed by CUDA events on its
 * stream.  vpmc_get_timing synchronises, returns accumulated milliseconds and launch counts per class
 * (0 beam_kernel: the persistent range-shifter / brass kernels S2-S3, 1 voxel_kernel S4-S7 incl. the influence pilot,
 * 2 dose conversion / uncertainty passes S6, 3 CSR writer passes S8, 4 the one-thread-per-item stage kernels: source +
 * opening phase S1/S3, aperture entry, CT entry, 5 the optimiser-iteration kernels S:8f-1) and resets. */
#define VPMC_N_KERNEL_CLASSES 6
int vpmc_set_timing(vpmc_t *h, int on);
int vpmc_get_timing(vpmc_t *h, double *ms_out, uint64_t *launches_out);

/* Measurement (S:8d (iii)): ceiling of global fp32 RED throughput on this device -- about n_ops atomicAdd(float) to
 * pseudo-random elements of a buffer of buffer_bytes (a power of two; 4 MB stays L2-resident), issued by one resident wave of
 * threads.  Returns the kernel's duration (CUDA events) and the exact number of REDs issued; bench.py reports the dose
 * scorer's RED rate against it.  Synchronous, default stream. */
int vpmc_bench_red(vpmc_t *h, uint64_t buffer_bytes, uint64_t n_ops, double *ms_out, uint64_t *n_ops_out);

/* Number of kernel launches issued by this handle so far (bench.py's gpu_launches). */
int vpmc_get_launch_count(vpmc_t *h, uint64_t *out);

const char *vpmc_last_error(const vpmc_t *h);
const char *vpmc_version(void);

#ifdef __cplusplus
}
#endif
#endif /* VPMC_H_ */
