// vpmc_kernels.cuh -- the sm_100a kernels of the hot path.  See DESIGN.md 5:
//   source_kernel     S1 (+ the opening phase of S3 for beams without range shifter): one thread per work item
//   beam_kernel<0>    S2: persistent warps carry histories through the range shifter; free lanes load the next record
//   ap_entry_kernel   S3, opening phase of the histories that left the range shifter, one thread per record
//   beam_kernel<1>    S3: persistent warps, brass steps of the aperture region; survivors are pushed to the CT queue
//   entry_kernel      CT entry (fp64), one thread per survivor
//   voxel_kernel      S4-S7: persistent warps pull survivors from the queue, step through the voxels and score;
//                     MODE 0 the dose grid(s), MODE 1 per-column boxes + overflow list, MODE 2 only column bounding boxes
//   dose_finalize / uncertainty kernels: S6 dose conversion and the C6 batch estimator
//   csr_* kernels     S8: threshold + count + scan + emit of the per-spot sparse columns
#pragma once
#include "vpmc_transport.cuh"

namespace vpk {

// work item -> (spot, history id, column / batch)   (C2)
struct WorkMap {
    int mode;                         // 0 dose, 1 influence
    unsigned long long n_items;       // items of this launch
    // dose: entry e = batch * n_spots + spot; cum[e] = first item of the entry, first[e] = its first history id
    const unsigned long long *cum;
    const unsigned long long *first;
    int n_entries, n_spots;
    // influence: item k -> local column k / n_sub, history i = k % n_sub of global spot cols[c] (or g0 + c)
    unsigned int hps, n_sub;
    const int *cols;
    int g0;
    // sequential batches (vpmc_dose_to_uncertainty): the high word of every history id = *batch_hi (D:R15); NULL = 0
    const unsigned int *batch_hi;
};

// influence-mode scoring target (S7): per-column private box in CT index space
struct ColumnBoxes {
    const int4 *lo;          // [n_cols] box low corner (ix, iy, iz, 0)
    const int4 *dim;         // [n_cols] box extent (bx, by, bz, 0)
    const unsigned long long *offset;   // [n_cols] offset of the box in `scratch`
    float *scratch;          // concatenated boxes (MeV)
    int *bbox;               // [n_cols][6] MODE 2: bounding box of all deposits; MODE 1: of the outside deposits that did
                             // NOT fit the overflow list (such a column is replayed with a larger box)
    // MODE 1: deposits outside the box go to a list of (column << 32 | voxel, MeV) entries, merged into the rows later
    unsigned long long *ovf_key;
    float *ovf_val;
    unsigned int *ovf_count;
    unsigned int ovf_cap;
};

__device__ __forceinline__ unsigned lanemask_lt()
{
    unsigned m; asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m)); return m;
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// item -> (global spot, history id, column or batch)
__device__ __forceinline__ void map_item(const WorkMap &wm, unsigned long long k, int &g, unsigned long long &hid, int &col)
{
    if (wm.mode == 0) {
        int lo = 0, hi = wm.n_entries;           // largest e with cum[e] <= k (empty entries are skipped by the search)
        while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (__ldg(wm.cum + mid) <= k) lo = mid; else hi = mid; }
        col = lo / wm.n_spots;                   // batch
        g = lo - col * wm.n_spots;
        hid = __ldg(wm.first + lo) + (k - __ldg(wm.cum + lo));
        if (wm.batch_hi) hid |= (unsigned long long)(*wm.batch_hi) << 32;
    } else {
        const unsigned long long c = k / wm.n_sub;
        col = (int)c;
        g = wm.cols ? __ldg(wm.cols + c) : wm.g0 + (int)c;
        hid = (unsigned long long)g * wm.hps + (k - c * wm.n_sub);
    }
}

// ------------------------------------------------------------------------------------------- scorers (S6, S7)
// S:8f-4, coarse-grid scoring: deposits can be scored on a grid whose cells are div[0] x div[1] x div[2] CT voxels
// (vpmc_set_scoring_grid); on = 0 is the plain case, scoring cell = CT voxel.
struct ScoreGeom { int on; int dx, dy, dz; int snx, sny; };

__device__ __forceinline__ void score_coords(const ScoreGeom &sg, const Hist &h, int &x, int &y, int &z)
{
    x = (int)h.g0; y = (int)h.g1; z = (int)h.g2;
    if (sg.on) { x /= sg.dx; y /= sg.dy; z /= sg.dz; }
}

struct DoseScorer {            // MODE 0: E_dep[batch][v] += dE, fp32 RED into L2-resident grids
    float *edep; unsigned long long nvox; ScoreGeom sg;
    __device__ __forceinline__ void begin(const Hist &) {}
    __device__ __forceinline__ void deposit(const Hist &h, float dep)
    {
        unsigned int v = h.g3;
        if (sg.on) { int x, y, z; score_coords(sg, h, x, y, z); v = (unsigned)(x + sg.snx * (y + sg.sny * z)); }
        atomicAdd(edep + (size_t)h.col * nvox + v, dep);
    }
    __device__ __forceinline__ void end(const Hist &) {}
    __device__ __forceinline__ void attach(int) {}
    __device__ __forceinline__ void room(int) {}
    __device__ __forceinline__ void finish(int) {}
};

__device__ __forceinline__ void bbox_merge(int *bb, int x0, int y0, int z0, int x1, int y1, int z1)
{
    atomicMin(bb + 0, x0); atomicMin(bb + 1, y0); atomicMin(bb + 2, z0);
    atomicMax(bb + 3, x1); atomicMax(bb + 4, y1); atomicMax(bb + 5, z1);
}

// MODE 1 appends a deposit outside its column's box to the overflow list.  One returning atomicAdd on the list's counter
// per such deposit (0.12 % of the steps) made the lane -- and with it the warp -- wait for a round trip to ONE contended L2
// address: a quarter of the kernel's stall samples.  Instead a warp reserves a STRETCH of kOvfStretch slots with one global
// atomic and hands them out through a cursor in shared memory; room() (all lanes, in the refill pass of the step loop) reserves
// the next stretch when fewer than kOvfRoom slots are left and fills what it abandons with sentinel keys (column 0xffffffff:
// skipped by the list's consumers), finish() does the same at the end of the kernel.  A deposit that finds no slot (nothing
// reserved yet, or more outside deposits in one step than were left) takes the global atomic as before.
constexpr unsigned int kOvfStretch = 64, kOvfRoom = 16;
constexpr unsigned long long kOvfSentinel = ~0ull;
constexpr int kOvfWarps = 8;              // = kBlock / 32 of the voxel kernel (static_assert there)

// this warp's stretch of the overflow list, in shared memory: [0] next slot, [1] end.  Found through the thread index where it
// is needed (rare paths) instead of being carried: the MODE 1 kernel has no register to spare.
__device__ __forceinline__ unsigned int *ovf_warp_state()
{
    __shared__ unsigned int s_ovf[kOvfWarps][2];
    return s_ovf[threadIdx.x >> 5];
}

// The two rare paths are kept out of line: inlined, their registers cost the step loop its constants (the kernel re-loaded
// them from the constant bank every pass: +30 instructions per step, measured).
// (arguments by value: a reference to the scorer's ColumnBoxes would put the struct on the local stack)
__device__ __noinline__ void ovf_append(unsigned long long *ovf_key, float *ovf_val, unsigned int *ovf_count, unsigned int ovf_cap, int *bbox,
                                        int c, unsigned int v, float dep, int sx, int sy, int sz)
{
    unsigned int *ws = ovf_warp_state();
    unsigned int slot = atomicAdd(ws, 1u);
    if (slot >= ws[1]) slot = atomicAdd(ovf_count, 1u);
    if (slot < ovf_cap) { ovf_key[slot] = ((unsigned long long)(unsigned)c << 32) | v; ovf_val[slot] = dep; }
    else bbox_merge(bbox + 6 * c, sx, sy, sz, sx, sy, sz);
}

__device__ __noinline__ void ovf_reserve(unsigned long long *ovf_key, float *ovf_val, unsigned int *ovf_count, unsigned int ovf_cap, int lane)   // all 32 lanes
{
    unsigned int *ws = ovf_warp_state();
    const unsigned int nxt = ws[0], end = ws[1];
    for (unsigned int i = min(nxt, end) + lane; i < end; i += 32)
        if (i < ovf_cap) { ovf_key[i] = kOvfSentinel; ovf_val[i] = 0.0f; }
    unsigned int base = 0;
    if (lane == 0) base = atomicAdd(ovf_count, kOvfStretch);
    base = __shfl_sync(0xffffffffu, base, 0);
    __syncwarp();
    if (lane == 0) { ws[0] = base; ws[1] = base + kOvfStretch; }
    __syncwarp();
}

struct BoxScorer {             // MODE 1: per-column private box; a deposit outside it goes to the overflow list
    ColumnBoxes cb; ScoreGeom sg;
    // the history's column box, read once when the lane takes the history (three dependent loads per deposit otherwise:
    // ncu long_scoreboard 2.2 against 0.5 in dose mode): low corner, extent, element offset of the box
    int lx, ly, lz, dx, dy, dz;
    unsigned long long off;
    __device__ __forceinline__ void begin(const Hist &h)
    {
        const int4 lo = __ldg(cb.lo + h.col), dm = __ldg(cb.dim + h.col);
        lx = lo.x; ly = lo.y; lz = lo.z; dx = dm.x; dy = dm.y; dz = dm.z;
        off = __ldg(cb.offset + h.col);
    }
    __device__ __forceinline__ void deposit(const Hist &h, float dep)
    {
        int sx, sy, sz;
        score_coords(sg, h, sx, sy, sz);
        const int bx = sx - lx, by = sy - ly, bz = sz - lz;
        if ((unsigned)bx < (unsigned)dx && (unsigned)by < (unsigned)dy && (unsigned)bz < (unsigned)dz)
            atomicAdd(cb.scratch + off + (bx + (unsigned long long)dx * (by + (unsigned long long)dy * bz)), dep);
        else ovf_append(cb.ovf_key, cb.ovf_val, cb.ovf_count, cb.ovf_cap, cb.bbox, h.col, sg.on ? (unsigned)(sx + sg.snx * (sy + sg.sny * sz)) : h.g3, dep, sx, sy, sz);
    }
    __device__ __forceinline__ void end(const Hist &) {}
    __device__ __forceinline__ void attach(int lane) { unsigned int *ws = ovf_warp_state(); if (lane < 2) ws[lane] = 0u; __syncwarp(); }
    __device__ __forceinline__ void room(int lane)             // all 32 lanes
    {
        const unsigned int *ws = ovf_warp_state();
        const unsigned int nxt = ws[0], end = ws[1];
        if (nxt + kOvfRoom <= end || (nxt | end) == 0u) return; // enough slots left, or no outside deposit so far
        ovf_reserve(cb.ovf_key, cb.ovf_val, cb.ovf_count, cb.ovf_cap, lane);
    }
    __device__ __forceinline__ void finish(int lane)           // closes the stretch the warp still holds
    {
        __syncwarp();
        const unsigned int *ws = ovf_warp_state();
        for (unsigned int i = min(ws[0], ws[1]) + lane; i < ws[1]; i += 32)
            if (i < cb.ovf_cap) { cb.ovf_key[i] = kOvfSentinel; cb.ovf_val[i] = 0.0f; }
    }
};

struct BoundsScorer {          // MODE 2 (pilot): bounding box of the deposits of each column
    int *bbox; ScoreGeom sg;
    int x0, y0, z0, x1, y1, z1;
    __device__ __forceinline__ void begin(const Hist &) { x0 = y0 = z0 = 0x7fffffff; x1 = y1 = z1 = -1; }
    __device__ __forceinline__ void deposit(const Hist &h, float)
    {
        int sx, sy, sz;
        score_coords(sg, h, sx, sy, sz);
        x0 = min(x0, sx); y0 = min(y0, sy); z0 = min(z0, sz);
        x1 = max(x1, sx); y1 = max(y1, sy); z1 = max(z1, sz);
    }
    __device__ __forceinline__ void end(const Hist &h) { if (x1 >= 0) bbox_merge(bbox + 6 * h.col, x0, y0, z0, x1, y1, z1); }
    __device__ __forceinline__ void attach(int) {}
    __device__ __forceinline__ void room(int) {}
    __device__ __forceinline__ void finish(int) {}
};

template <int MODE> struct ScorerOf;
template <> struct ScorerOf<0> { typedef DoseScorer type; };
template <> struct ScorerOf<1> { typedef BoxScorer type; };
template <> struct ScorerOf<2> { typedef BoundsScorer type; };

struct ScoreArgs { float *edep; unsigned long long nvox; ColumnBoxes cb; ScoreGeom sg; };

template <int MODE> __device__ __forceinline__ typename ScorerOf<MODE>::type make_scorer(const ScoreArgs &a);
template <> __device__ __forceinline__ DoseScorer make_scorer<0>(const ScoreArgs &a) { return DoseScorer{ a.edep, a.nvox, a.sg }; }
template <> __device__ __forceinline__ BoxScorer make_scorer<1>(const ScoreArgs &a) { BoxScorer s; s.cb = a.cb; s.sg = a.sg; s.lx = s.ly = s.lz = 0; s.dx = s.dy = s.dz = 0; s.off = 0ull; return s; }
template <> __device__ __forceinline__ BoundsScorer make_scorer<2>(const ScoreArgs &a) { BoundsScorer s; s.bbox = a.cb.bbox; s.sg = a.sg; return s; }

// ------------------------------------------------------------------------------------------- S1-S7
// Pipeline of one chunk of work items:
//   source_kernel  one thread per item: item -> spot, history id; S1 sampling; writes a 48-byte source record
//   beam_kernel    persistent warps step histories through range shifter and aperture; a free lane is refilled by
//                  LOADING the next source record (cheap, so lanes are refilled eagerly); survivors -> queue
//   entry_kernel   one thread per survivor: beam frame -> CT frame, ray-box entry (fp64), record rewritten in place
//   voxel_kernel   persistent warps step survivors through the voxels and score; refill = loading a record
// The expensive once-per-history work (Philox + accurate log / sincos of the source, the fp64 CT entry) runs in plain
// fully converged kernels; the persistent kernels contain nothing but the step loop.
constexpr int kBlock = 256;
constexpr int kWarps = kBlock / 32;
#ifndef VPK_REFILL_MIN
#define VPK_REFILL_MIN 6
#endif
constexpr int kRefillMin = VPK_REFILL_MIN;   // S6b: free lanes are refilled once at least this many of a warp's lanes are free

#ifndef VPK_MIN_BLOCKS
#define VPK_MIN_BLOCKS 4
#endif

// range-shifter input records of a chunk (histories on the entrance plane of the range shifter: direction +w, nothing
// accumulated yet), SoA of 16-byte words
struct SourceBuf {
    uint4 *s0;    // x hi, x lo, y hi, y lo (beam frame, fp32 pairs)
    uint4 *s1;    // E, tau_star, col | beam << 24, step
    uint4 *s2;    // R lo, R hi, hid_lo, hid_hi
    unsigned int *count;   // records written
};

// Histories handed from one stage to the next: SoA of 16-byte records (80 B per history, 96 B with q5), written and read
// coalesced.  Three queues per chunk: range shifter -> aperture entry; aperture entry -> aperture kernel (with q5); CT queue.
// Beam-line stages write the beam-frame state; entry_kernel rewrites q0 (and the direction) of the CT queue as the CT state.
struct Queue {
    uint4 *q0;    // beam frame: x hi, x lo, y hi, y lo;  CT: local x, y, z (fp32), voxel index (0xffffffff = missed the CT)
    float4 *q1;   // ux, uy, uz, E
    float4 *q2;   // lx, ly, lz, t_rad
    uint4 *q3;    // tau, tau_star, step, col | beam << 24
    uint4 *q4;    // R lo, R hi, hid_lo, hid_hi
    float4 *q5;   // aperture queue only: brass budget (h.rx), depth inside the aperture region (h.rz), -, -
    unsigned int *count;   // entries pushed
    unsigned int *head;    // entries claimed by the consuming persistent kernel
    unsigned int capacity;
};

// slot of this lane in a queue: one atomic per warp.  Must be called by all 32 lanes.
__device__ __forceinline__ unsigned int warp_push_slot(unsigned int *counter, bool want, int lane)
{
    const unsigned m = __ballot_sync(0xffffffffu, want);
    if (m == 0u) return 0u;
    unsigned base = 0;
    const int leader = __ffs(m) - 1;
    if (lane == leader) base = atomicAdd(counter, (unsigned)__popc(m));
    base = __shfl_sync(0xffffffffu, base, leader);
    return base + (unsigned)__popc(m & lanemask_lt());
}

// Slot of this thread's record with ONE atomic per block: with one per warp, a chunk of 2^23 records sends 2.6e5 atomics to
// the same address, and the L2 serialises those (source_kernel: its incident-energy and record-count atomics were its whole
// run time).  Worth it only where the block's warps arrive together -- behind divergent work the barrier costs more than
// the atomics (measured in ap_entry_kernel).  Must be called by all threads of the block, once per kernel.
__device__ __forceinline__ unsigned int block_push_slot(unsigned int *counter, bool want)
{
    __shared__ unsigned int s_cnt[kWarps];
    __shared__ unsigned int s_base;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned int m = __ballot_sync(0xffffffffu, want);
    if (lane == 0) s_cnt[warp] = (unsigned)__popc(m);
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned int run = 0;
#pragma unroll
        for (int w = 0; w < kWarps; ++w) { const unsigned int c = s_cnt[w]; s_cnt[w] = run; run += c; }
        s_base = run ? atomicAdd(counter, run) : 0u;
    }
    __syncthreads();
    return s_base + s_cnt[warp] + (unsigned)__popc(m & lanemask_lt());
}

// block sum of a double in a fixed order, valid in thread 0.  Must be called by all threads of the block, once per kernel.
__device__ __forceinline__ double block_sum_thread0(double v)
{
    __shared__ double s_v[kWarps];
    v = warp_sum(v);
    if ((threadIdx.x & 31) == 0) s_v[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int w = 0; w < kWarps; ++w) t += s_v[w];
    }
    return t;
}

__device__ __forceinline__ void queue_store(const Queue &q, unsigned int slot, const Hist &h)
{
    if (slot >= q.capacity) return;
    q.q0[slot] = make_uint4(h.g0, h.g1, h.g2, h.g3);
    q.q1[slot] = make_float4(h.ux, h.uy, h.uz, h.E);
    q.q2[slot] = make_float4(h.lx, h.ly, h.lz, h.t_rad);
    q.q3[slot] = make_uint4(__float_as_uint(h.tau), __float_as_uint(h.tau_star), h.step, (unsigned)h.col | ((unsigned)(h.region >> 8) << 24));
    const unsigned long long rb = (unsigned long long)__double_as_longlong(h.R);
    q.q4[slot] = make_uint4((unsigned)rb, (unsigned)(rb >> 32), h.hid_lo, h.hid_hi);
    if (q.q5) q.q5[slot] = make_float4(h.rx, h.rz, 0.0f, 0.0f);
}

// beam-frame record -> history standing in region `reg` (REG_TO_AP after the range shifter, REG_AP from the aperture queue)
__device__ __forceinline__ void queue_load_beam(const Queue &q, unsigned int slot, int reg, float c_log, Hist &h)
{
    const uint4 p0 = q.q0[slot];
    const float4 a = q.q1[slot], b = q.q2[slot];
    const uint4 e = q.q3[slot], f = q.q4[slot];
    h.g0 = p0.x; h.g1 = p0.y; h.g2 = p0.z; h.g3 = p0.w;
    h.ux = a.x; h.uy = a.y; h.uz = a.z; h.E = a.w;
    h.lx = b.x; h.ly = b.y; h.lz = b.z; h.t_rad = b.w; h.f_rad = highland_f(b.w, c_log);
    h.tau = __uint_as_float(e.x); h.tau_star = __uint_as_float(e.y); h.step = e.z;
    h.col = (int)(e.w & 0xffffffu); h.region = reg | (int)((e.w >> 24) << 8);
    h.R = __longlong_as_double((long long)(((unsigned long long)f.y << 32) | f.x));
    h.hid_lo = f.z; h.hid_hi = f.w;
    h.rx = 0.0f; h.ry = 0.0f; h.rz = 0.0f;
    if (q.q5) { const float4 g = q.q5[slot]; h.rx = g.x; h.rz = g.y; }
}

// per-warp flush of the tallies: lane counters into the warp's shared slots, then <= 13 global atomics per warp
__device__ __forceinline__ void flush_warp_tallies(WarpTally *w, const LaneCounters &lc, DevTallies *tal, int lane)
{
    const double inc = warp_sum(lc.incident);
    const unsigned nct = __reduce_add_sync(0xffffffffu, lc.n_ct), ndev = __reduce_add_sync(0xffffffffu, lc.n_dev);
    const unsigned nslab = __reduce_add_sync(0xffffffffu, lc.n_slab);
    __syncwarp();
    if (lane == 0) { w->d[TD_INCIDENT] += inc; w->c[TC_STEPS_CT] += nct; w->c[TC_STEPS_DEV] += ndev; w->c[TC_STEPS_SLAB] += nslab; }
    __syncwarp();
    if (lane < TD_N && w->d[lane] != 0.0) atomicAdd(&tal->incident + lane, w->d[lane]);
    if (lane < TC_N && w->c[lane]) atomicAdd(&tal->n_stopped_ct + lane, (unsigned long long)w->c[lane]);
}

// a history that ended as ESCAPED in one of the one-thread-per-history kernels (u_w <= 0 in the beam line: never with the
// closed-form physics at these energies, kept for the rule of C4): booked with plain warp-reduced atomics
__device__ __forceinline__ void book_escapes_converged(DevTallies *tal, bool esc, float E, unsigned int steps)
{
    const unsigned m = __ballot_sync(0xffffffffu, esc);
    if (m == 0u) return;
    const double e = warp_sum(esc ? (double)E : 0.0);
    const unsigned n_dev = __reduce_add_sync(0xffffffffu, esc ? steps : 0u);
    if ((threadIdx.x & 31) == 0) {
        atomicAdd(&tal->escaped, e);
        atomicAdd(&tal->n_escaped, (unsigned long long)__popc(m));
        atomicAdd(&tal->n_steps_dev, (unsigned long long)n_dev);
    }
}

// S1 + the converged part of S3: items [item0, item0 + n) -> sampled histories, each routed to the stage it needs next:
//   beam with a range shifter        -> range-shifter input record (on its entrance plane);
//   aperture only, clean transit     -> CT queue (the whole opening phase of P:L87 runs here, converged);
//   aperture only, brass step due    -> aperture queue;
//   no device                        -> CT queue.
__global__ void __launch_bounds__(kBlock)
source_kernel(const Ctx c, const WorkMap wm, const unsigned long long item0, const float4 *__restrict__ spots,
              const double *__restrict__ spot_R0, const int *__restrict__ spot_beam, const SourceBuf sb, const Queue q_ap,
              const Queue q_ct, DevTallies *tal)
{
    const unsigned long long k = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    double inc = 0.0;
    int dest = 0;                      // 1 range shifter, 2 aperture queue, 3 CT queue, 4 escaped
    Hist h;
    h.E = 0.0f; h.step = 0u; h.region = 0;
    int reg = -1;
    NullTracer tr;
    if (k < wm.n_items) {
        int g; unsigned long long hid;
        map_item(wm, item0 + k, g, hid, h.col);
        h.hid_lo = (uint32_t)hid; h.hid_hi = (uint32_t)(hid >> 32);
        const int beam = __ldg(spot_beam + g);
        sample_source(c.P, c.beams[beam], beam, __ldg(spots + g), __ldg(spot_R0 + g), h, c.K);
        inc = (double)h.E;
        reg = h.region & 0xff;
        if (reg == REG_TO_RS) dest = (rs_enter(c, h, tr) == BEAM_CONT) ? 1 : 4;
    }
    // Up to here every warp of the block has done the same work: the range-shifter records and the incident energy are
    // pushed with one atomic per BLOCK (block_push_slot, block_sum_thread0).  The opening phase below is divergent -- a barrier
    // behind it would make every warp wait for the block's slowest -- so the two queues it feeds keep one atomic per warp.
    const unsigned s_rs = block_push_slot(sb.count, dest == 1);
    inc = block_sum_thread0(inc);
    if (threadIdx.x == 0 && inc != 0.0) atomicAdd(&tal->incident, inc);
    if (dest == 1) {
        const unsigned long long rb = (unsigned long long)__double_as_longlong(h.R);
        sb.s0[s_rs] = make_uint4(h.g0, h.g1, h.g2, h.g3);
        sb.s1[s_rs] = make_uint4(__float_as_uint(h.E), __float_as_uint(h.tau_star), (unsigned)h.col | ((unsigned)(h.region >> 8) << 24), h.step);
        sb.s2[s_rs] = make_uint4((unsigned)rb, (unsigned)(rb >> 32), h.hid_lo, h.hid_hi);
    }
    if (reg == REG_TO_AP) { const int st = ap_enter(c, h, tr); dest = (st == BEAM_EXIT) ? 3 : (st == BEAM_CONT ? 2 : 4); }
    else if (reg >= 0 && reg != REG_TO_RS) dest = 3;
    const unsigned s_ap = warp_push_slot(q_ap.count, dest == 2, lane);
    const unsigned s_ct = warp_push_slot(q_ct.count, dest == 3, lane);
    if (dest == 2) queue_store(q_ap, s_ap, h);
    else if (dest == 3) queue_store(q_ct, s_ct, h);
    book_escapes_converged(tal, dest == 4, h.E, h.step);
}

// Aperture entry of the histories that left the range shifter, one thread per record: vacuum drift to the aperture
// entrance and the opening phase (ap_enter) -> CT queue (clean transit, or no aperture) | aperture queue (brass step due)
__global__ void __launch_bounds__(kBlock)
ap_entry_kernel(const Ctx c, const Queue q_in, const Queue q_ap, const Queue q_ct, DevTallies *tal)
{
    const unsigned n_q = min(*q_in.count, q_in.capacity);
    const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    int dest = 0;
    Hist h;
    h.E = 0.0f; h.step = 0u;
    if (i < n_q) {
        queue_load_beam(q_in, i, REG_TO_AP, c.P.c_log, h);
        if (__ldg(&c.beams[h.region >> 8].has_ap)) {
            NullTracer tr;
            const int st = ap_enter(c, h, tr);
            dest = (st == BEAM_EXIT) ? 3 : (st == BEAM_CONT ? 2 : 4);
        } else { h.region = REG_TO_CT | (h.region & ~0xff); dest = 3; }
    }
    const unsigned s_ap = warp_push_slot(q_ap.count, dest == 2, lane);
    const unsigned s_ct = warp_push_slot(q_ct.count, dest == 3, lane);
    if (dest == 2) queue_store(q_ap, s_ap, h);
    else if (dest == 3) queue_store(q_ct, s_ct, h);
    book_escapes_converged(tal, dest == 4, h.E, h.step);
}

// S2 / S3: persistent warps; every lane carries one history through ONE device -- STAGE 0 the range shifter (input: the
// range-shifter records), STAGE 1 the brass of the aperture region (input: the aperture queue).  A lane whose history ended
// or left the device loads the next record (warp-aggregated claim on the input counter); histories that left the device
// alive are pushed to `out` (STAGE 0: the aperture-entry queue, STAGE 1: the CT queue) with one atomic per warp and pass.
template <int STAGE, int FL>
__global__ void __launch_bounds__(kBlock, VPK_MIN_BLOCKS)
beam_kernel(const Ctx c, const SourceBuf sb, const Queue in, const Queue out, unsigned int *head, DevTallies *tal)
{
    __shared__ WarpTally wt_all[kWarps];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x < kWarps * (int)(sizeof(WarpTally) / 4)) reinterpret_cast<unsigned int *>(wt_all)[threadIdx.x] = 0u;
    __syncthreads();
    NullTracer tr;
    LaneCounters lc;
    Hist h;
    h.region = REG_TO_CT; h.col = 0; h.step = 0u; h.E = 0.0f; h.R = 0.0;
    float dep = 0.0f;                      // energy deposited in this device so far
    const unsigned int n_items = (STAGE == 0) ? *sb.count : min(*in.count, in.capacity);
    int pend = BEAM_CONT;                  // status of a finished history whose bookkeeping is still due
    bool alive = false, exhausted = false;
    for (;;) {
        // S6b, event pass: once enough lanes are free, book their finished histories, push the survivors to the queue and
        // load the next records -- all of it converged over those lanes
        const unsigned free_mask = __ballot_sync(0xffffffffu, !alive);
        const unsigned pend_mask = __ballot_sync(0xffffffffu, !alive && pend != BEAM_CONT);
        const int n_free = __popc(free_mask);
        if ((n_free >= kRefillMin || n_free == 32) && (!exhausted || pend_mask)) {
            const bool push = !alive && pend == BEAM_EXIT;
            const unsigned slot = warp_push_slot(out.count, push, lane);
            if (push) queue_store(out, slot, h);
            book_beam_end(c.P, h, !alive && pend != BEAM_CONT, pend, dep, STAGE == 0 ? TD_DEP_RS : TD_DEP_BRASS, lc, wt_all + warp, lane);
            pend = alive ? pend : BEAM_CONT;
            if (!exhausted) {
                unsigned base = 0;
                const int leader = __ffs(free_mask) - 1;
                if (lane == leader) base = atomicAdd(head, (unsigned)n_free);
                base = __shfl_sync(0xffffffffu, base, leader);
                exhausted = base + (unsigned)n_free >= n_items;
                if (!alive) {
                    const unsigned k = base + __popc(free_mask & lanemask_lt());
                    if (k < n_items) {
                        if (STAGE == 0) {
                            const uint4 a = sb.s0[k], b = sb.s1[k], e = sb.s2[k];
                            h.g0 = a.x; h.g1 = a.y; h.g2 = a.z; h.g3 = a.w;
                            h.rx = 0.0f; h.ry = 0.0f; h.rz = 0.0f;
                            h.E = __uint_as_float(b.x); h.tau_star = __uint_as_float(b.y);
                            h.col = (int)(b.z & 0xffffffu); h.region = REG_RS | (int)((b.z >> 24) << 8);
                            h.step = b.w;
                            h.R = __longlong_as_double((long long)(((unsigned long long)e.y << 32) | e.x));
                            h.hid_lo = e.z; h.hid_hi = e.w;
                            h.tau = 0.0f; h.t_rad = 0.0f; h.f_rad = 1.0f;
                            h.ux = 0.0f; h.uy = 0.0f; h.uz = 1.0f; h.lx = 0.0f; h.ly = 0.0f; h.lz = 0.0f;
                        } else queue_load_beam(in, k, REG_AP, c.P.c_log, h);
                        dep = 0.0f;
                        alive = true;
                    }
                }
            }
        }
        const unsigned alive_mask = __ballot_sync(0xffffffffu, alive);
        if (alive_mask == 0u) {
            if (exhausted && !__any_sync(0xffffffffu, pend != BEAM_CONT)) break;
            continue;
        }
        if (alive) {
            const int status = (STAGE == 0) ? rs_iter<FL>(c, h, dep, lc, tr) : ap_iter<FL>(c, h, dep, lc, tr, alive_mask);
            if (status != BEAM_CONT) { alive = false; pend = status; }
        }
    }
    flush_warp_tallies(wt_all + warp, lc, tal, lane);
}

// CT entry of the survivors (C3), one thread per queue entry: q0 becomes (local x, y, z, voxel index) and the direction
// the CT-frame direction.  A history that misses the CT box is booked as ESCAPED and its record marked.
__global__ void __launch_bounds__(kBlock)
entry_kernel(const Ctx c, const Queue q, DevTallies *tal)
{
    const unsigned n_q = min(*q.count, q.capacity);
    const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
    double esc = 0.0; unsigned n_esc = 0, n_dev = 0;
    if (i < n_q) {
        Hist h;
        const uint4 p0 = q.q0[i];
        const float4 a = q.q1[i], b = q.q2[i];
        const uint4 e = q.q3[i];
        h.g0 = p0.x; h.g1 = p0.y; h.g2 = p0.z; h.g3 = p0.w;
        h.ux = a.x; h.uy = a.y; h.uz = a.z; h.E = a.w;
        h.lx = b.x; h.ly = b.y; h.lz = b.z;
        h.step = e.z; h.hid_lo = 0u; h.hid_hi = 0u;
        const DevBeam *bp = c.beams + (e.w >> 24);
        const float w_now = bp->has_ap ? bp->w_ap_out : (bp->has_rs ? bp->w_rs_out : bp->w_start);
        NullTracer tr;
        const int ec = enter_ct(c, *bp, w_now, h, tr);
        n_dev = h.step;
        if (ec != CONT) { esc = (double)h.E; n_esc = 1u; h.g3 = 0xffffffffu; }
        q.q0[i] = make_uint4(__float_as_uint(h.rx), __float_as_uint(h.ry), __float_as_uint(h.rz), h.g3);
        q.q1[i] = make_float4(h.ux, h.uy, h.uz, a.w);
        q.q2[i] = make_float4(h.lx, h.ly, h.lz, b.w);
        q.q3[i] = make_uint4(e.x, e.y, h.step, e.w);
    }
    // the drift-step count is booked once per block (every warp has some: one same-address atomic per warp otherwise);
    // escapes are rare and stay per warp
    __shared__ unsigned int s_dev[kWarps];
    esc = warp_sum(esc);
    n_esc = __reduce_add_sync(0xffffffffu, n_esc); n_dev = __reduce_add_sync(0xffffffffu, n_dev);
    if ((threadIdx.x & 31) == 0) {
        s_dev[threadIdx.x >> 5] = n_dev;
        if (esc != 0.0) atomicAdd(&tal->escaped, esc);
        if (n_esc) atomicAdd(&tal->n_escaped, (unsigned long long)n_esc);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long t = 0;
#pragma unroll
        for (int w = 0; w < kWarps; ++w) t += s_dev[w];
        if (t) atomicAdd(&tal->n_steps_dev, t);
    }
}

// S4-S7: persistent warps; free lanes load survivors from the queue (one atomic per warp and refill) and step through
// the voxels with ct_step().  MODE 0 scores the dose grid(s), MODE 1 per-column boxes, MODE 2 only column bounding
// boxes.  SMEM_LUT: material table staged in shared memory.
template <int MODE, bool SMEM_LUT, int FL>
__global__ void __launch_bounds__(kBlock, VPK_MIN_BLOCKS)
voxel_kernel(const Ctx c, const Queue q, const float4 *__restrict__ lut_g, const ScoreArgs sa, DevTallies *tal)
{
    extern __shared__ float4 smem4[];
    WarpTally *wt_all = reinterpret_cast<WarpTally *>(smem4);
    float4 *lut_s = smem4 + (kWarps * sizeof(WarpTally) + 15) / 16;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x < kWarps * (int)(sizeof(WarpTally) / 4)) reinterpret_cast<unsigned int *>(wt_all)[threadIdx.x] = 0u;
    if (SMEM_LUT)
        for (int i = threadIdx.x; i < c.G.n_lut; i += blockDim.x) lut_s[i] = lut_g[i];
    __syncthreads();
    typename ScorerOf<MODE>::type sc = make_scorer<MODE>(sa);
    static_assert(kOvfWarps == kWarps, "one stretch of the overflow list per warp of the block");
    sc.attach(lane);                                       // MODE 1: the warp's (empty) stretch of the overflow list
    NullTracer tr;
    LaneCounters lc;
    Hist h;
    h.region = REG_CT; h.col = 0; h.step = 0u;
    float hdep = 0.0f;
    int hu_pre = 0;                    // HU of the voxel the lane's history stands in (fetched ahead of the step that needs it)
    const unsigned n_q = min(*q.count, q.capacity);
    const unsigned nxy = (unsigned)(c.G.nx * c.G.ny);
    int pend = CONT;                       // cause of a finished history whose bookkeeping is still due
    bool alive = false, exhausted = false;
    for (;;) {
        // S6b, event pass (see beam_kernel)
        const unsigned free_mask = __ballot_sync(0xffffffffu, !alive);
        const unsigned pend_mask = __ballot_sync(0xffffffffu, !alive && pend != CONT);
        const int n_free = __popc(free_mask);
        if ((n_free >= kRefillMin || n_free == 32) && (!exhausted || pend_mask)) {
            sc.room(lane);
            if (!alive && pend != CONT) sc.end(h);
            book_ct_end(c.P, h, !alive && pend != CONT, pend, hdep, wt_all + warp, lane);
            pend = alive ? pend : CONT;
            if (!exhausted) {
                unsigned base = 0;
                const int leader = __ffs(free_mask) - 1;
                if (lane == leader) base = atomicAdd(q.head, (unsigned)n_free);
                base = __shfl_sync(0xffffffffu, base, leader);
                exhausted = base + (unsigned)n_free >= n_q;
                if (!alive) {
                    const unsigned slot = base + __popc(free_mask & lanemask_lt());
                    if (slot < n_q) {
                        const uint4 p0 = q.q0[slot];
                        if (p0.w != 0xffffffffu) {
                            const float4 a = q.q1[slot], b = q.q2[slot];
                            const uint4 e = q.q3[slot], f = q.q4[slot];
                            h.rx = __uint_as_float(p0.x); h.ry = __uint_as_float(p0.y); h.rz = __uint_as_float(p0.z);
                            h.g3 = p0.w;
                            h.g2 = p0.w / nxy;
                            const unsigned rem = p0.w - h.g2 * nxy;
                            h.g1 = rem / (unsigned)c.G.nx; h.g0 = rem - h.g1 * (unsigned)c.G.nx;
                            h.ux = a.x; h.uy = a.y; h.uz = a.z; h.E = a.w;
                            h.lx = b.x; h.ly = b.y; h.lz = b.z; h.t_rad = b.w; h.f_rad = highland_f(b.w, c.P.c_log);
                            h.tau = __uint_as_float(e.x); h.tau_star = __uint_as_float(e.y); h.step = e.z;
                            h.col = (int)(e.w & 0xffffffu); h.region = REG_CT | (int)((e.w >> 24) << 8);
                            h.R = __longlong_as_double((long long)(((unsigned long long)f.y << 32) | f.x));
                            h.hid_lo = f.z; h.hid_hi = f.w;
                            hdep = 0.0f;
                            hu_pre = (int)__ldg(c.hu + h.g3);
                            sc.begin(h);
                            alive = true;
                        }
                    }
                }
            }
        }
        if (!__any_sync(0xffffffffu, alive)) {
            if (exhausted && !__any_sync(0xffffffffu, pend != CONT)) break;
            continue;
        }
        if (alive) {
            int cause;
            if (SMEM_LUT) cause = ct_step<FL>(c, LutShared{ lut_s }, h, hdep, lc, sc, tr, &hu_pre);
            else cause = ct_step<FL>(c, LutGlobal{ lut_g }, h, hdep, lc, sc, tr, &hu_pre);
            if (cause != CONT) { alive = false; pend = cause; }
            else hu_pre = (int)__ldg(c.hu + h.g3);            // the next step's voxel: in flight during the refill pass and the face distances
        }
    }
    sc.finish(lane);
    flush_warp_tallies(wt_all + warp, lc, tal, lane);
}

// S0 for polygon openings (S:8f-2): classify the cells of the coarse grid over the polygon's bounding box.  Every point of a
// cell lies within half a diagonal of its centre, so when the centre is farther than that from the boundary the whole cell
// is on the centre's side, and around ANY point of the cell the answer holds within d - half_diag (Euclidean), i.e. within
// (d - half_diag) / sqrt(2) in the L-infinity norm the step loop measures its lateral travel in.
__global__ void polygon_grid_kernel(const float2 *__restrict__ poly, int n, int nx, int ny, float x0, float y0, float cell, float *__restrict__ grid)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nx * ny) return;
    const int iy = t / nx, ix = t - iy * nx;
    float d2;
    const bool in = polygon_query(poly, n, fmaf((float)ix + 0.5f, cell, x0), fmaf((float)iy + 0.5f, cell, y0), d2);
    const float d = sqrtf(d2);
    const float half_diag = 0.70711f * cell * 1.01f + 1e-4f;        // + the rounding of the cell lookup
    float v = 0.0f;
    if (d > half_diag) { const float r = fmaxf(0.7f * (d - half_diag), 1e-6f); v = in ? r : -r; }
    grid[t] = v;
}

// ------------------------------------------------------------------------------------------- trace (test-only)
// one thread per selected history, from the source to its end through the SAME step functions as the production kernels;
// records (RecTracer) or a digest (DigestTracer) per history
template <class Tracer>
__device__ __forceinline__ float trace_history(const Ctx &c, unsigned long long hid, int g, const float4 *spots, const double *spot_R0,
                                               const int *spot_beam, const float4 *lut_g, Tracer &tr)
{
    Hist h; LaneCounters lc; NullScorer sc; NullSink sink;
    float hdep = 0.0f;
    h.col = 0;
    h.hid_lo = (uint32_t)hid; h.hid_hi = (uint32_t)(hid >> 32);
    const int beam = spot_beam[g];
    sample_source(c.P, c.beams[beam], beam, spots[g], spot_R0[g], h, c.K);
    int code = BEAM_CONT;
    float dep_rs = 0.0f, dep_ap = 0.0f;
    for (int it = 0; it < 1000000 && code == BEAM_CONT; ++it) code = beam_step(c, h, dep_rs, dep_ap, lc, tr);
    if (code == BEAM_EXIT && ct_entry(c, h, lc, sink, tr) == CONT) {
        for (int it = 0; it < 1000000; ++it)
            if (ct_step<-1>(c, LutGlobal{ lut_g }, h, hdep, lc, sc, tr) != CONT) break;
    }
    return hdep;
}

__global__ void trace_kernel(const Ctx c, const unsigned long long *__restrict__ hids, const int *__restrict__ spot_of, int n,
                             const float4 *__restrict__ spots, const double *__restrict__ spot_R0,
                             const int *__restrict__ spot_beam, const float4 *__restrict__ lut_g,
                             StepRec *recs, int max_steps, int *nrec)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    RecTracer tr{ recs + (size_t)i * max_steps, max_steps, 0 };
    const int g = spot_of[i];
    if (g < 0) { nrec[i] = 0; return; }
    trace_history(c, hids[i], g, spots, spot_R0, spot_beam, lut_g, tr);
    nrec[i] = tr.n;
}

// digests of the contiguous history ids [hid0, hid0 + n) of a dose-mode run: spot by search in the id prefix `start`
__global__ void digest_kernel(const Ctx c, unsigned long long hid0, int n, const unsigned long long *__restrict__ start, int n_spots,
                              const float4 *__restrict__ spots, const double *__restrict__ spot_R0,
                              const int *__restrict__ spot_beam, const float4 *__restrict__ lut_g, Digest *__restrict__ out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const unsigned long long hid = hid0 + (unsigned long long)i;
    int lo = 0, hi = n_spots;                    // largest g with start[g] <= hid (empty spots are skipped by the search)
    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (start[mid] <= hid) lo = mid; else hi = mid; }
    DigestTracer tr;
    tr.start(hid);
    tr.d.dep_ct = trace_history(c, hid, lo, spots, spot_R0, spot_beam, lut_g, tr);
    out[i] = tr.d;
}

// ------------------------------------------------------------------------------------------- one step from a state (test-only)
struct StateIn {    // == vpmc_state
    unsigned long long hid;
    int kind, step, beam, spot;
    int ivox[3];
    int pad_;
    double r[3], u[3];
    double E, t_rad, tau, tau_star;
};
struct StateOut {   // == vpmc_state_out
    int region, cause, step_after, n_steps;
    int ivox_after[3];
    int pad_;
    double r[3], u[3];
    double E, R, s, dep, t_rad, tau, tau_star;
};
enum : int { STEP_SOURCE = 0, STEP_DRIFT_TO_RS, STEP_RS, STEP_DRIFT_TO_AP, STEP_AP, STEP_CT_ENTRY, STEP_CT };

// Runs the SAME step functions as the production kernels (sample_source, drift_gap, beam_step, ct_entry, ct_step) once,
// from a state given in fp64 and converted to the kernel's own representation (fp64 range from E, hi + lo direction and
// beam-frame position, voxel + local offset).
__global__ void step_state_kernel(const Ctx c, const StateIn *__restrict__ in, int n, const float4 *__restrict__ spots,
                                  const double *__restrict__ spot_R0, const float4 *__restrict__ lut_g, StateOut *__restrict__ out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const StateIn q = in[i];
    const DevBeam &b = c.beams[q.beam];
    const DevGrid &G = c.G;
    StepRec rec;
    RecTracer tr{ &rec, 1, 0 };
    Hist h; LaneCounters lc; NullScorer sc; NullSink sink;
    StateOut o;
    memset(&o, 0, sizeof(o));
    h.col = 0;
    h.hid_lo = (uint32_t)q.hid; h.hid_hi = (uint32_t)(q.hid >> 32);
    if (q.kind == STEP_SOURCE) {
        sample_source(c.P, b, q.beam, spots[q.spot], spot_R0[q.spot], h, c.K);
        o.region = REG_VAC; o.cause = CONT;
        o.r[0] = beam_x(h); o.r[1] = beam_y(h); o.r[2] = (double)b.w_start;
        o.u[2] = 1.0;
        o.E = (double)h.E; o.R = h.R; o.tau_star = (double)h.tau_star;
        out[i] = o;
        return;
    }
    h.E = (float)q.E;
    h.R = (double)c.P.alpha * pow(q.E, (double)c.P.p);
    h.t_rad = (float)q.t_rad; h.f_rad = highland_f(h.t_rad, c.P.c_log);
    h.tau = (float)q.tau; h.tau_star = (float)q.tau_star;
    h.step = (uint32_t)q.step;
    h.ux = (float)q.u[0]; h.uy = (float)q.u[1]; h.uz = (float)q.u[2];
    h.lx = (float)(q.u[0] - (double)h.ux); h.ly = (float)(q.u[1] - (double)h.uy); h.lz = (float)(q.u[2] - (double)h.uz);
    h.rx = h.ry = h.rz = 0.0f;
    float dep_rs = 0.0f, dep_ap = 0.0f, hdep = 0.0f;
    if (q.kind != STEP_CT) { set_beam_x(h, q.r[0]); set_beam_y(h, q.r[1]); }
    if (q.kind == STEP_DRIFT_TO_RS || q.kind == STEP_DRIFT_TO_AP) {
        const bool rs = q.kind == STEP_DRIFT_TO_RS;
        const float w1 = rs ? b.w_rs_in : b.w_ap_in;
        const float w0 = rs ? b.w_start : (b.has_rs ? b.w_rs_out : b.w_start);
        h.region = (rs ? REG_TO_RS : REG_TO_AP) | (q.beam << 8);
        const int cause = drift_gap(h, w1 - w0, w1, tr);
        if (cause != CONT) { rec.region = REG_VAC; rec.cause = ESCAPED; rec.s = 0.0f; tr.n = 1; }
        o.r[0] = beam_x(h); o.r[1] = beam_y(h); o.r[2] = (cause == CONT) ? (double)w1 : q.r[2];
    } else if (q.kind == STEP_RS || q.kind == STEP_AP) {
        const bool rs = q.kind == STEP_RS;
        const float w_in = rs ? b.w_rs_in : b.w_ap_in;
        h.region = (rs ? REG_RS : REG_AP) | (q.beam << 8);
        h.rz = (float)(q.r[2] - (double)w_in);
        beam_step(c, h, dep_rs, dep_ap, lc, tr);
        if (tr.n == 1) { o.r[0] = beam_x(h); o.r[1] = beam_y(h); o.r[2] = (double)w_in + (double)h.rz; }
        else { o.r[0] = (double)rec.r[0]; o.r[1] = (double)rec.r[1]; o.r[2] = (double)rec.r[2]; }
    } else if (q.kind == STEP_CT_ENTRY) {
        h.region = REG_TO_CT | (q.beam << 8);
        ct_entry(c, h, lc, sink, tr);
    } else {
        h.region = REG_CT | (q.beam << 8);
        const double lo[3] = { (double)G.ox, (double)G.oy, (double)G.oz }, hh[3] = { (double)G.hx, (double)G.hy, (double)G.hz };
        float l[3];
        for (int a = 0; a < 3; ++a) l[a] = (float)fmin(fmax(q.r[a] - fma((double)q.ivox[a], hh[a], lo[a]), 0.0), hh[a]);
        h.rx = l[0]; h.ry = l[1]; h.rz = l[2];
        h.g0 = (uint32_t)q.ivox[0]; h.g1 = (uint32_t)q.ivox[1]; h.g2 = (uint32_t)q.ivox[2];
        h.g3 = (uint32_t)(q.ivox[0] + G.nx * (q.ivox[1] + G.ny * q.ivox[2]));
        ct_step<-1>(c, LutGlobal{ lut_g }, h, hdep, lc, sc, tr);
    }
    if (q.kind == STEP_CT_ENTRY || q.kind == STEP_CT) {
        o.ivox_after[0] = (int)h.g0; o.ivox_after[1] = (int)h.g1; o.ivox_after[2] = (int)h.g2;
        if (rec.cause == ESCAPED && q.kind == STEP_CT_ENTRY) { o.r[0] = (double)rec.r[0]; o.r[1] = (double)rec.r[1]; o.r[2] = (double)rec.r[2]; }
        else {
            o.r[0] = fma((double)(int)h.g0, (double)G.hx, (double)G.ox) + (double)h.rx;
            o.r[1] = fma((double)(int)h.g1, (double)G.hy, (double)G.oy) + (double)h.ry;
            o.r[2] = fma((double)(int)h.g2, (double)G.hz, (double)G.oz) + (double)h.rz;
        }
    }
    o.region = rec.region; o.cause = rec.cause; o.n_steps = tr.n; o.s = (double)rec.s;
    const bool one = tr.n == 1;
    o.step_after = one ? (int)h.step : q.step + 1;
    o.u[0] = one ? (double)h.ux + (double)h.lx : q.u[0];
    o.u[1] = one ? (double)h.uy + (double)h.ly : q.u[1];
    o.u[2] = one ? (double)h.uz + (double)h.lz : q.u[2];
    o.E = one ? (double)h.E : q.E;
    o.R = h.R;
    o.dep = (double)(dep_rs + dep_ap + hdep);
    o.t_rad = one ? (double)h.t_rad : q.t_rad;
    o.tau = one ? (double)h.tau : q.tau;
    o.tau_star = (double)h.tau_star;
    out[i] = o;
}

// ------------------------------------------------------------------------------------------- S6 / C6
// Density in the dose conversion: max(rho_v, rho_min) of the voxel, or, with coarse-grid scoring, the sum of that over the
// cell's voxels (cell_rho, built by cell_rho_kernel): dose of a cell = its energy / its mass.
__device__ __forceinline__ float score_density(const float *__restrict__ cell_rho, const short *__restrict__ hu, const float4 *__restrict__ lut,
                                               int hu_min, int n_lut, float rho_min, long long v)
{
    if (cell_rho) return __ldg(cell_rho + v);
    int t = (int)__ldg(hu + v) - hu_min;
    t = min(max(t, 0), n_lut - 1);
    return fmaxf(__ldg(lut + t).y, rho_min);
}

__global__ void cell_rho_kernel(const short *__restrict__ hu, const float4 *__restrict__ lut, DevGrid G, float rho_min, ScoreGeom sg, int snz,
                                float *__restrict__ cell_rho)
{
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= (long long)sg.snx * sg.sny * snz) return;
    const int cz = (int)(c / ((long long)sg.snx * sg.sny)), rem = (int)(c - (long long)cz * sg.snx * sg.sny), cy = rem / sg.snx, cx = rem - cy * sg.snx;
    float sum = 0.0f;
    for (int z = cz * sg.dz; z < min((cz + 1) * sg.dz, G.nz); ++z)
        for (int y = cy * sg.dy; y < min((cy + 1) * sg.dy, G.ny); ++y)
            for (int x = cx * sg.dx; x < min((cx + 1) * sg.dx, G.nx); ++x)
                sum += score_density(nullptr, hu, lut, G.hu_min, G.n_lut, rho_min, x + (long long)G.nx * (y + (long long)G.ny * z));
    cell_rho[c] = sum;
}

// One pass over the B batch grids: dose[v] = coef * sum_b E_b[v] / max(rho_v, rho_min); with B >= 2 also the batch
// sums s1 = sum_b f_b E_b, s2 = sum_b (f_b E_b)^2 (f_b = N / N_b scales a batch to full weight) for C6.
__global__ void dose_finalize_kernel(const float *__restrict__ edep, int B, const float *__restrict__ fb,
                                     const short *__restrict__ hu, const float4 *__restrict__ lut, DevGrid G, float rho_min,
                                     float coef, float *__restrict__ dose, float *__restrict__ s1, float *__restrict__ s2,
                                     long long n, unsigned int *max_bits, const float *__restrict__ cell_rho)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    float mx = 0.0f;
    for (long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x; v < n; v += stride) {
        float sum = 0.0f, a1 = 0.0f, a2 = 0.0f;
        for (int b = 0; b < B; ++b) {
            const float x = edep[(size_t)b * n + v];
            sum += x;
            const float y = __ldg(fb + b) * x;
            a1 += y; a2 = fmaf(y, y, a2);
        }
        const float rho = score_density(cell_rho, hu, lut, G.hu_min, G.n_lut, rho_min, v);
        const float dv = __fdiv_rn(coef * sum, rho);
        dose[v] = dv;
        if (s1) { s1[v] = a1; s2[v] = a2; }
        mx = fmaxf(mx, dv);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    if ((threadIdx.x & 31) == 0 && mx > 0.0f) atomicMax(max_bits, __float_as_uint(mx));
}

// C6: mean over voxels with dose >= 0.5 max of sigma_v / Dbar_v, from s1 = sum_b D_b, s2 = sum_b D_b^2 (raw MeV
// scale cancels; the density factor is per-voxel constant and cancels too)
__global__ void uncertainty_kernel(const float *__restrict__ dose, const float *__restrict__ s1,
                                   const float *__restrict__ s2, long long n, int B, const unsigned int *max_bits,
                                   double *acc /* [0] sum of rel sigma, [1] count */)
{
    const float half_max = 0.5f * __uint_as_float(*max_bits);
    const long long stride = (long long)gridDim.x * blockDim.x;
    double s = 0.0, c = 0.0;
    for (long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x; v < n; v += stride) {
        if (dose[v] >= half_max && dose[v] > 0.0f) {
            const double a = (double)s1[v], b = (double)s2[v];
            const double mean = a / B;
            double var = (b - a * a / B) / ((double)B * (B - 1));
            if (var < 0.0) var = 0.0;
            s += sqrt(var) / mean;
            c += 1.0;
        }
    }
    s = warp_sum(s); c = warp_sum(c);
    if ((threadIdx.x & 31) == 0 && c > 0.0) { atomicAdd(acc, s); atomicAdd(acc + 1, c); }
}

// ------------------------------------------------------------------------------------------- S:8f-3: on-GPU stopping rule
// Sequential batches (SURVEY.md 8(d) metric 2, "<0.5 %"): after every batch the C6 estimator over the batches so
// far decides on the DEVICE whether another batch runs -- the batch pass is the body of a CUDA-graph WHILE node whose
// condition seq_decide_kernel sets, so the host enqueues one graph and never looks at intermediate results.
// With equal batches the estimator needs only s1 = sum_b E_b and s2 = sum_b E_b^2 per voxel.
struct SeqState {
    unsigned int batch;        // batches finished so far = index of the batch in flight
    unsigned int max_bits;     // bits of max_v s1[v] (monotone: s1 only grows)
    float unc;                 // estimate after the last finished batch (0 while < 2 batches)
    unsigned int stopped_by_target;
    double acc[2];             // sum of sigma_v / mean_v, number of voxels
};

__global__ void seq_accumulate_kernel(float *__restrict__ edep, float *__restrict__ s1, float *__restrict__ s2, long long n, SeqState *st)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    float mx = 0.0f;
    for (long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x; v < n; v += stride) {
        const float e = edep[v];
        if (e != 0.0f) { edep[v] = 0.0f; s2[v] = fmaf(e, e, s2[v]); }
        const float a = s1[v] + e;
        if (e != 0.0f) s1[v] = a;
        mx = fmaxf(mx, a);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    if ((threadIdx.x & 31) == 0 && mx > 0.0f) atomicMax(&st->max_bits, __float_as_uint(mx));
}

// C6 over the B = st->batch + 1 batches finished once this pass runs: mean over voxels with s1 >= 0.5 max of sigma_v / mean_v
__global__ void seq_uncertainty_kernel(const float *__restrict__ s1, const float *__restrict__ s2, long long n, SeqState *st)
{
    const int B = (int)st->batch + 1;
    if (B < 2) return;
    const float half_max = 0.5f * __uint_as_float(st->max_bits);
    const long long stride = (long long)gridDim.x * blockDim.x;
    double s = 0.0, c = 0.0;
    for (long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x; v < n; v += stride) {
        const float a1 = s1[v];
        if (a1 >= half_max && a1 > 0.0f) {
            const double a = (double)a1, b = (double)s2[v];
            double var = (b - a * a / B) / ((double)B * (B - 1));
            if (var < 0.0) var = 0.0;
            s += sqrt(var) / (a / B);
            c += 1.0;
        }
    }
    s = warp_sum(s); c = warp_sum(c);
    if ((threadIdx.x & 31) == 0 && c > 0.0) { atomicAdd(&st->acc[0], s); atomicAdd(&st->acc[1], c); }
}

// one thread: close the batch, decide whether the WHILE node runs its body again
__global__ void seq_decide_kernel(cudaGraphConditionalHandle handle, SeqState *st, int min_batches, int max_batches, float target)
{
    const int B = (int)(st->batch += 1u);
    const float unc = (B >= 2 && st->acc[1] > 0.0) ? (float)(st->acc[0] / st->acc[1]) : 0.0f;
    st->unc = unc;
    st->acc[0] = 0.0; st->acc[1] = 0.0;
    const bool reached = B >= 2 && B >= min_batches && st->max_bits != 0u && unc <= target;
    st->stopped_by_target = reached ? 1u : 0u;
    cudaGraphSetConditional(handle, (reached || B >= max_batches) ? 0u : 1u);
}

// dose[v] = coef_batch / B * s1[v] / max(rho_v, rho_min), coef_batch = (W / N_b) / V * 1.602e-10 (C6 with N = B N_b)
__global__ void seq_finalize_kernel(const float *__restrict__ s1, const short *__restrict__ hu, const float4 *__restrict__ lut, DevGrid G,
                                    float rho_min, float coef_batch, const SeqState *st, float *__restrict__ dose, long long n,
                                    const float *__restrict__ cell_rho)
{
    const float coef = coef_batch / (float)max(st->batch, 1u);
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x; v < n; v += stride)
        dose[v] = __fdiv_rn(coef * s1[v], score_density(cell_rho, hu, lut, G.hu_min, G.n_lut, rho_min, v));
}

// ------------------------------------------------------------------------------------------- S8: CSR writer
// A "column" is a dense fp32 box (lo, dim) of the CT grid stored contiguously at scratch + offset, element
// e = bx + dim.x (by + dim.y bz), so ascending e is ascending voxel index v.  Columns are cut into tiles of kTile
// elements; tile t of the launch belongs to the column found by binary search in tile0[] (prefix of tiles per column).
// Passes: (1) convert E_dep -> dose value and take the column maximum; (2) count the kept entries per tile
// (val > 0 and val >= rel_thr * max, product in fp32); (3) per column: exclusive scan of its tile counts;
// (4) emit (voxel index, value) at base[c] + tile_off + rank.  vpmc_csr_from_dense runs (1) without the conversion on a
// single column of shape (n, 1, 1), so the writer the tests pin bit-exactly is the writer the influence path uses.
constexpr int kTile = 2048;
constexpr int kPerThread = kTile / kBlock;

struct CsrCols {
    const int4 *lo, *dim;
    const unsigned long long *offset;   // element offset of each column in `data`
    const int *tile0;                   // [n_cols + 1] prefix of tiles per column
    const int *skip;                    // [n_cols] or NULL: non-zero = column not written in this round
    const int *tile_col;                // [n_tiles] or NULL: column of every tile (the passes would otherwise each spend a
                                        // dependent 11-load binary search per 8 KB tile: measured 2.4 TB/s instead of HBM speed)
    int n_cols, n_tiles;
    int nx, ny;                         // of the CT grid (voxel index of box element)
};

__device__ __forceinline__ int tile_column(const CsrCols &cc, int tile)
{
    if (cc.tile_col) return __ldg(cc.tile_col + tile);       // looked up once per group by csr_tile_cols_kernel
    int lo = 0, hi = cc.n_cols;
    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (__ldg(cc.tile0 + mid) <= tile) lo = mid; else hi = mid; }
    return lo;
}

// column of every tile, once per group
__global__ void csr_tile_cols_kernel(CsrCols cc, int *__restrict__ tile_col)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= cc.n_tiles) return;
    cc.tile_col = nullptr;
    tile_col[t] = tile_column(cc, t);
}

// first element of this thread in its tile (a box has < 2^31 elements) and the number of elements it owns (0..kPerThread)
__device__ __forceinline__ int tile_thread_range(const CsrCols &cc, int tile, int c, const int4 dm, unsigned int &e)
{
    const unsigned int vol = (unsigned int)dm.x * (unsigned int)dm.y * (unsigned int)dm.z;
    e = (unsigned int)(tile - __ldg(cc.tile0 + c)) * kTile + threadIdx.x * kPerThread;
    if (e >= vol) return 0;
    const unsigned int left = vol - e;
    return left < (unsigned)kPerThread ? (int)left : kPerThread;
}
// box coordinates of element e (two 32-bit divisions: only taken by threads that need a voxel index)
__device__ __forceinline__ void box_decode(unsigned int e, const int4 dm, int &bx, int &by, int &bz)
{
    const unsigned int row = e / (unsigned)dm.x;
    bx = (int)(e - row * (unsigned)dm.x);
    bz = (int)(row / (unsigned)dm.y);
    by = (int)(row - (unsigned)bz * (unsigned)dm.y);
}
__device__ __forceinline__ void box_next(const int4 dm, int &bx, int &by, int &bz)
{
    if (++bx == dm.x) { bx = 0; if (++by == dm.y) { by = 0; ++bz; } }
}
// voxel indices of the thread's kPerThread consecutive elements from e on, for boxes at least kPerThread wide: the first
// nrow lie in e's row (vA + i), the others in the next row (vB + i); no per-element carry chain
struct BoxRun { int vA, vB, nrow; };
__device__ __forceinline__ BoxRun box_run(const CsrCols &cc, unsigned int e, const int4 lo, const int4 dm)
{
    int bx, by, bz;
    box_decode(e, dm, bx, by, bz);
    BoxRun r;
    r.vA = (lo.x + bx) + cc.nx * ((lo.y + by) + cc.ny * (lo.z + bz));
    r.nrow = dm.x - bx;
    if (++by == dm.y) { by = 0; ++bz; }
    r.vB = lo.x + cc.nx * ((lo.y + by) + cc.ny * (lo.z + bz)) - r.nrow;      // beyond the box only for elements beyond cnt (never kept)
    return r;
}
// the thread's kPerThread = 8 consecutive elements: two 16-byte loads when it owns all eight and they are aligned (always
// the case inside a box: offsets and tiles are multiples of 8 elements), element-wise otherwise; missing elements read 0
__device__ __forceinline__ void load8(const float *p, int cnt, float x[kPerThread])
{
    static_assert(kPerThread == 8, "load8 assumes 8 elements per thread");
    if (cnt == kPerThread && (reinterpret_cast<size_t>(p) & 15) == 0) {
        const float4 a = *reinterpret_cast<const float4 *>(p), b = *reinterpret_cast<const float4 *>(p + 4);
        x[0] = a.x; x[1] = a.y; x[2] = a.z; x[3] = a.w; x[4] = b.x; x[5] = b.y; x[6] = b.z; x[7] = b.w;
    } else {
#pragma unroll
        for (int i = 0; i < kPerThread; ++i) x[i] = (i < cnt) ? p[i] : 0.0f;
    }
}

template <bool CONVERT>
__global__ void __launch_bounds__(kBlock)
csr_max_kernel(const CsrCols cc, float *__restrict__ data, const short *__restrict__ hu, const float4 *__restrict__ lut,
               int hu_min, int n_lut, float rho_min, float coef, unsigned int *__restrict__ colmax_bits, const float *__restrict__ cell_rho)
{
    for (int tile = blockIdx.x; tile < cc.n_tiles; tile += gridDim.x) {
        const int c = tile_column(cc, tile);
        if (cc.skip && __ldg(cc.skip + c)) continue;
        const int4 lo = __ldg(cc.lo + c), dm = __ldg(cc.dim + c);
        unsigned int e;
        const int cnt = tile_thread_range(cc, tile, c, dm, e);
        float *p = data + __ldg(cc.offset + c) + e;
        float x[kPerThread];
        load8(p, cnt, x);
        float mx = 0.0f;
        bool any = false;
#pragma unroll
        for (int i = 0; i < kPerThread; ++i) any = any || (x[i] != 0.0f);
        if (CONVERT && any) {
            if (dm.x >= kPerThread) {
                const BoxRun br = box_run(cc, e, lo, dm);
#pragma unroll
                for (int i = 0; i < kPerThread; ++i)
                    if (x[i] != 0.0f)
                        x[i] = __fdiv_rn(coef * x[i], score_density(cell_rho, hu, lut, hu_min, n_lut, rho_min, (long long)((i < br.nrow ? br.vA : br.vB) + i)));
            } else {
                int bx, by, bz;
                box_decode(e, dm, bx, by, bz);
#pragma unroll
                for (int i = 0; i < kPerThread; ++i) {
                    if (x[i] != 0.0f) {
                        const long long v = (lo.x + bx) + (long long)cc.nx * ((lo.y + by) + (long long)cc.ny * (lo.z + bz));
                        x[i] = __fdiv_rn(coef * x[i], score_density(cell_rho, hu, lut, hu_min, n_lut, rho_min, v));
                    }
                    box_next(dm, bx, by, bz);
                }
            }
            if (cnt == kPerThread && (reinterpret_cast<size_t>(p) & 15) == 0) {
                *reinterpret_cast<float4 *>(p) = make_float4(x[0], x[1], x[2], x[3]);
                *reinterpret_cast<float4 *>(p + 4) = make_float4(x[4], x[5], x[6], x[7]);
            } else {
                for (int i = 0; i < cnt; ++i) p[i] = x[i];
            }
        }
#pragma unroll
        for (int i = 0; i < kPerThread; ++i) mx = fmaxf(mx, x[i]);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        if ((threadIdx.x & 31) == 0 && mx > 0.0f) atomicMax(colmax_bits + c, __float_as_uint(mx));
    }
}

__device__ __forceinline__ bool csr_keep(float x, float thr) { return x > 0.0f && x >= thr; }

__global__ void __launch_bounds__(kBlock)
csr_count_kernel(const CsrCols cc, const float *__restrict__ data, const unsigned int *__restrict__ colmax_bits, float rel_thr,
                 unsigned int *__restrict__ tile_count)
{
    __shared__ unsigned int wsum[kWarps];
    for (int tile = blockIdx.x; tile < cc.n_tiles; tile += gridDim.x) {
        const int c = tile_column(cc, tile);
        unsigned int k = 0;
        if (!(cc.skip && __ldg(cc.skip + c))) {
            const int4 dm = __ldg(cc.dim + c);
            unsigned int e;
            const int cnt = tile_thread_range(cc, tile, c, dm, e);
            const float thr = rel_thr * __uint_as_float(__ldg(colmax_bits + c));
            float x[kPerThread];
            load8(data + __ldg(cc.offset + c) + e, cnt, x);
#pragma unroll
            for (int i = 0; i < kPerThread; ++i) k += csr_keep(x[i], thr) ? 1u : 0u;
        }
        k = __reduce_add_sync(0xffffffffu, k);
        if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = k;
        __syncthreads();
        if (threadIdx.x == 0) {
            unsigned int s = 0;
#pragma unroll
            for (int w = 0; w < kWarps; ++w) s += wsum[w];
            tile_count[tile] = s;
        }
        __syncthreads();
    }
}

// one block per column: exclusive scan of the column's tile counts (in place) and the column total
__global__ void __launch_bounds__(kBlock)
csr_tile_scan_kernel(const CsrCols cc, unsigned int *__restrict__ tile_count, long long *__restrict__ col_nnz)
{
    __shared__ unsigned int wsum[kWarps];
    __shared__ unsigned int carry_s;
    const int c = blockIdx.x;
    const int t0 = __ldg(cc.tile0 + c), t1 = __ldg(cc.tile0 + c + 1);
    if (threadIdx.x == 0) carry_s = 0u;
    __syncthreads();
    for (int base = t0; base < t1; base += kBlock) {
        const int t = base + threadIdx.x;
        const unsigned int x = (t < t1) ? tile_count[t] : 0u;
        unsigned int inc = x;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const unsigned int y = __shfl_up_sync(0xffffffffu, inc, o); if ((threadIdx.x & 31) >= o) inc += y; }
        if ((threadIdx.x & 31) == 31) wsum[threadIdx.x >> 5] = inc;
        __syncthreads();
        unsigned int woff = 0;
        for (int w = 0; w < (int)(threadIdx.x >> 5); ++w) woff += wsum[w];
        const unsigned int carry = carry_s;
        if (t < t1) tile_count[t] = carry + woff + inc - x;
        __syncthreads();
        if (threadIdx.x == kBlock - 1) carry_s = carry + woff + inc;
        __syncthreads();
    }
    if (threadIdx.x == 0) col_nnz[c] = (cc.skip && __ldg(cc.skip + c)) ? 0ll : (long long)carry_s;
}

// Pass 4.  A warp owns kTile / kWarps = 256 consecutive elements of the tile and takes them as 8 rows of 32, lane l the
// element 32 i + l of row i: the loads are 128-byte rows, and -- the point -- the kept entries of a row go to CONSECUTIVE
// output positions (rank by ballot), so a store instruction fills whole 32-byte sectors.  With 8 consecutive elements per
// thread (as in passes 1 and 2, where only the loads matter) a warp's store touched up to 32 sectors for 4 bytes each:
// 10x the written bytes in L2 write traffic (lts__t_bytes 4.0e11 against pass 2's 1.5e11 for the same reads).
__global__ void __launch_bounds__(kBlock)
csr_emit_kernel(const CsrCols cc, const float *__restrict__ data, const unsigned int *__restrict__ colmax_bits, float rel_thr,
                const unsigned int *__restrict__ tile_off, const long long *__restrict__ col_base,
                int *__restrict__ out_idx, float *__restrict__ out_val)
{
    constexpr int kRows = kTile / kWarps / 32;
    __shared__ unsigned int wsum[kWarps];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned int lt = (1u << lane) - 1u;
    for (int tile = blockIdx.x; tile < cc.n_tiles; tile += gridDim.x) {
        const int c = tile_column(cc, tile);
        if (cc.skip && __ldg(cc.skip + c)) continue;          // block-uniform
        const int4 lo = __ldg(cc.lo + c), dm = __ldg(cc.dim + c);
        const unsigned int vol = (unsigned int)dm.x * (unsigned int)dm.y * (unsigned int)dm.z;
        const unsigned int e_w = (unsigned int)(tile - __ldg(cc.tile0 + c)) * kTile + (unsigned int)warp * (kTile / kWarps);
        const float thr = rel_thr * __uint_as_float(__ldg(colmax_bits + c));
        const float *p = data + __ldg(cc.offset + c) + e_w + lane;
        float x[kRows];
#pragma unroll
        for (int i = 0; i < kRows; ++i) x[i] = (e_w + 32u * i + lane < vol) ? p[32 * i] : 0.0f;
        unsigned int bal[kRows], total = 0;
#pragma unroll
        for (int i = 0; i < kRows; ++i) { bal[i] = __ballot_sync(0xffffffffu, csr_keep(x[i], thr)); total += __popc(bal[i]); }
        if (lane == 0) wsum[warp] = total;
        __syncthreads();
        if (total) {                                           // warp-uniform
            unsigned int woff = 0;
            for (int w = 0; w < warp; ++w) woff += wsum[w];
            const long long pos0 = __ldg(col_base + c) + (long long)__ldg(tile_off + tile) + woff;
            int *oi = out_idx + pos0;
            float *ov = out_val + pos0;
            // box coordinates of the warp's first element, then row by row (+32) and lane by lane (+lane) with carries
            int bx, by, bz;
            box_decode(e_w < vol ? e_w : 0u, dm, bx, by, bz);
            unsigned int run = 0;
#pragma unroll
            for (int i = 0; i < kRows; ++i) {
                if (bal[i] >> lane & 1u) {
                    int ex = bx + lane, ey = by, ez = bz;
                    while (ex >= dm.x) { ex -= dm.x; if (++ey == dm.y) { ey = 0; ++ez; } }
                    const unsigned int pos = run + __popc(bal[i] & lt);
                    oi[pos] = (lo.x + ex) + cc.nx * ((lo.y + ey) + cc.ny * (lo.z + ez));
                    ov[pos] = x[i];
                }
                run += __popc(bal[i]);
                bx += 32;
                while (bx >= dm.x) { bx -= dm.x; if (++by == dm.y) { by = 0; ++bz; } }
            }
        }
        __syncthreads();
    }
}

// ---- overflow list (deposits outside a column's box): (column << 32 | cell, MeV) entries in arrival order.  They are
// bucketed by column (count -> offsets on the host -> scatter through a cursor per column), and then ONE CTA per column sorts
// its bucket by cell in shared memory, sums the deposits of a cell, converts to dose, folds the values into the column
// maximum, thresholds and writes the kept (cell, value) pairs, ascending, at the start of the column's own stretch of the
// staging arrays -- all hand-written; a bucket larger than kOvfSortCap is not handled here: the column is replayed with a
// larger box (the host sees the counts).
constexpr int kOvfSortCap = 16384;        // entries a CTA sorts in shared memory (128 KB)
constexpr int kOvfBlock = 1024;

__global__ void ovf_hist_kernel(const unsigned long long *__restrict__ key, unsigned int n, unsigned int *__restrict__ col_cnt)
{
    for (unsigned int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const unsigned c = (unsigned)(key[i] >> 32);
        if (c != 0xffffffffu) atomicAdd(col_cnt + c, 1u);       // not a sentinel (BoxScorer::close_stretch)
    }
}

// bounding box (scoring-grid coordinates) of the overflow entries of the columns flagged in `lost`
__global__ void ovf_bbox_kernel(const unsigned long long *__restrict__ key, unsigned int n, const int *__restrict__ lost, int snx, int sny, int *__restrict__ bbox)
{
    for (unsigned int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const unsigned c = (unsigned)(key[i] >> 32), v = (unsigned)key[i];
        if (c == 0xffffffffu || !__ldg(lost + c)) continue;
        const int z = (int)(v / (unsigned)(snx * sny)), rem = (int)(v - (unsigned)z * (unsigned)(snx * sny)), y = rem / snx, x = rem - y * snx;
        bbox_merge(bbox + 6 * c, x, y, z, x, y, z);
    }
}

__global__ void ovf_scatter_kernel(const unsigned long long *__restrict__ key, const float *__restrict__ val, unsigned int n,
                                   const unsigned int *__restrict__ col_off, unsigned int *__restrict__ cursor, unsigned int *__restrict__ b_cell,
                                   float *__restrict__ b_val)
{
    for (unsigned int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const unsigned long long k = key[i];
        const unsigned c = (unsigned)(k >> 32);
        if (c == 0xffffffffu) continue;
        const unsigned pos = __ldg(col_off + c) + atomicAdd(cursor + c, 1u);
        b_cell[pos] = (unsigned)k; b_val[pos] = val[i];
    }
}

// one CTA per column
__global__ void __launch_bounds__(kOvfBlock)
ovf_columns_kernel(const unsigned int *__restrict__ b_cell, const float *__restrict__ b_val, const unsigned int *__restrict__ col_off,
                   const unsigned int *__restrict__ col_cnt, const int *__restrict__ skip, const short *__restrict__ hu, const float4 *__restrict__ lut,
                   int hu_min, int n_lut, float rho_min, float coef, const float *__restrict__ cell_rho, float rel_thr,
                   unsigned int *__restrict__ colmax_bits, int *__restrict__ out_idx, float *__restrict__ out_val, unsigned int *__restrict__ kept_cnt,
                   unsigned int sort_cap)
{
    extern __shared__ unsigned int ovf_smem[];
    unsigned int *key = ovf_smem;
    float *val = reinterpret_cast<float *>(ovf_smem + kOvfSortCap);
    __shared__ unsigned int s_warp[kOvfBlock / 32];
    __shared__ unsigned int s_max, s_carry;
    const int c = blockIdx.x;
    const unsigned int n = __ldg(col_cnt + c), off = __ldg(col_off + c);
    if (threadIdx.x == 0) kept_cnt[c] = 0u;
    if (n == 0u || n > sort_cap || __ldg(skip + c)) return;
    unsigned int P = 1u;
    while (P < n) P <<= 1;
    for (unsigned int i = threadIdx.x; i < P; i += kOvfBlock) { key[i] = (i < n) ? b_cell[off + i] : 0xffffffffu; val[i] = (i < n) ? b_val[off + i] : 0.0f; }
    __syncthreads();
    // bitonic sort by cell
    for (unsigned int k = 2; k <= P; k <<= 1)
        for (unsigned int j = k >> 1; j > 0; j >>= 1) {
            for (unsigned int i = threadIdx.x; i < P; i += kOvfBlock) {
                const unsigned int l = i ^ j;
                if (l > i) {
                    const unsigned int a = key[i], b = key[l];
                    if ((a > b) == ((i & k) == 0u)) { key[i] = b; key[l] = a; const float t = val[i]; val[i] = val[l]; val[l] = t; }
                }
            }
            __syncthreads();
        }
    // the first entry of every cell sums the cell's deposits and converts them to dose; the others are marked
    if (threadIdx.x == 0) { s_max = __ldg(colmax_bits + c); s_carry = 0u; }
    __syncthreads();
    float mx = 0.0f;
    for (unsigned int i = threadIdx.x; i < n; i += kOvfBlock) {
        const unsigned int v = key[i];
        if (i > 0 && key[i - 1] == v) continue;
        float sum = val[i];
        for (unsigned int l = i + 1; l < n && key[l] == v; ++l) sum += val[l];
        const float x = __fdiv_rn(coef * sum, score_density(cell_rho, hu, lut, hu_min, n_lut, rho_min, (long long)v));
        mx = fmaxf(mx, x);
        val[i] = x;                                       // (heads only read their own run: no other thread reads val[i] as a head's input)
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    if ((threadIdx.x & 31) == 0 && mx > 0.0f) atomicMax(&s_max, __float_as_uint(mx));
    __syncthreads();
    const unsigned int cm = s_max;
    if (threadIdx.x == 0) colmax_bits[c] = cm;
    const float thr = rel_thr * __uint_as_float(cm);
    // keep and compact, in cell order
    for (unsigned int base = 0; base < n; base += kOvfBlock) {
        const unsigned int i = base + threadIdx.x;
        const bool head = i < n && (i == 0 || key[i - 1] != key[i]);
        const bool keep = head && csr_keep(val[i], thr);
        const unsigned int bal = __ballot_sync(0xffffffffu, keep);
        if ((threadIdx.x & 31) == 0) s_warp[threadIdx.x >> 5] = __popc(bal);
        __syncthreads();
        unsigned int woff = 0, tot = 0;
        for (int w = 0; w < kOvfBlock / 32; ++w) { const unsigned int t = s_warp[w]; if (w < (int)(threadIdx.x >> 5)) woff += t; tot += t; }
        const unsigned int carry = s_carry;
        if (keep) { const unsigned int pos = off + carry + woff + __popc(bal & lanemask_lt()); out_idx[pos] = (int)key[i]; out_val[pos] = val[i]; }
        __syncthreads();
        if (threadIdx.x == 0) s_carry = carry + tot;
        __syncthreads();
    }
    if (threadIdx.x == 0) kept_cnt[c] = s_carry;
}

// final assembly: row r = merge of its staged box entries (a) and its kept overflow entries (b), both ascending in voxel
// index and disjoint, into the scenario's CSR arrays.  Position of an element = its rank in its own list + the number of
// elements of the other list below it (binary search).
constexpr int kGatherStage = 8192;
__global__ void csr_gather_rows_kernel(int n_rows, const long long *__restrict__ src_off, const long long *__restrict__ ovf_off,
                                       const int *__restrict__ ovf_n, const long long *__restrict__ row_ptr,
                                       const int *__restrict__ s_idx, const float *__restrict__ s_val,
                                       const int *__restrict__ o_idx, const float *__restrict__ o_val,
                                       int *__restrict__ idx, float *__restrict__ val)
{
    __shared__ int s_o[kGatherStage];        // the row's overflow indices: the box elements' searches stay inside the SM
    for (int r = blockIdx.x; r < n_rows; r += gridDim.x) {
        const long long dst = __ldg(row_ptr + r), n = __ldg(row_ptr + r + 1) - dst, sa = __ldg(src_off + r);
        const int nb = __ldg(ovf_n + r);
        const long long na = n - nb, sb = __ldg(ovf_off + r);
        // four elements per thread in flight: with one, the copy ran at 1.8 TB/s (bytes in flight per SM / latency)
        if (nb == 0) {
            long long i = threadIdx.x;
            for (; i + 3 * blockDim.x < na; i += 4 * blockDim.x) {
                int v[4]; float x[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) { v[u] = __ldg(s_idx + sa + i + u * blockDim.x); x[u] = __ldg(s_val + sa + i + u * blockDim.x); }
#pragma unroll
                for (int u = 0; u < 4; ++u) { idx[dst + i + u * blockDim.x] = v[u]; val[dst + i + u * blockDim.x] = x[u]; }
            }
            for (; i < na; i += blockDim.x) { idx[dst + i] = s_idx[sa + i]; val[dst + i] = s_val[sa + i]; }
            continue;
        }
        if (nb <= kGatherStage) {
            __syncthreads();                  // the previous row's searches are done
            for (int j = threadIdx.x; j < nb; j += blockDim.x) s_o[j] = o_idx[sb + j];
            __syncthreads();
            long long i = threadIdx.x;
            for (; i + 3 * blockDim.x < na; i += 4 * blockDim.x) {
                int v[4]; float x[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) { v[u] = __ldg(s_idx + sa + i + u * blockDim.x); x[u] = __ldg(s_val + sa + i + u * blockDim.x); }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    int lo = 0, hi = nb;
                    while (lo < hi) { const int mid = (lo + hi) >> 1; if (s_o[mid] < v[u]) lo = mid + 1; else hi = mid; }
                    idx[dst + i + u * blockDim.x + lo] = v[u]; val[dst + i + u * blockDim.x + lo] = x[u];
                }
            }
            for (; i < na; i += blockDim.x) {
                const int v = s_idx[sa + i];
                const float x = s_val[sa + i];
                int lo = 0, hi = nb;
                while (lo < hi) { const int mid = (lo + hi) >> 1; if (s_o[mid] < v) lo = mid + 1; else hi = mid; }
                idx[dst + i + lo] = v; val[dst + i + lo] = x;
            }
        } else {
            for (long long i = threadIdx.x; i < na; i += blockDim.x) {
                const int v = s_idx[sa + i];
                int lo = 0, hi = nb;
                while (lo < hi) { const int mid = (lo + hi) >> 1; if (o_idx[sb + mid] < v) lo = mid + 1; else hi = mid; }
                idx[dst + i + lo] = v; val[dst + i + lo] = s_val[sa + i];
            }
        }
        for (int j = threadIdx.x; j < nb; j += blockDim.x) {
            const int v = o_idx[sb + j];
            long long lo = 0, hi = na;
            while (lo < hi) { const long long mid = (lo + hi) >> 1; if (s_idx[sa + mid] < v) lo = mid + 1; else hi = mid; }
            idx[dst + j + lo] = v; val[dst + j + lo] = o_val[sb + j];
        }
    }
}

}  // namespace vpk
