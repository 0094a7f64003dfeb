// vpmc_kernels.cuh -- the sm_100a kernels of the hot path and their launch-side
// descriptors.  See DESIGN.md 5 for the launch structure:
//   beamline_kernel   S1-S3: one thread per history; survivors are pushed (warp-aggregated) to a queue
//   voxel_kernel      S4-S6b: persistent warps pull histories from the queue, refill dead lanes, score
//   batch/dose/uncertainty kernels: S6 dose conversion and the C6 batch estimator
//   influence kernels S7-S8: per-column private sub-volumes, threshold + scan + CSR emit
#pragma once
#include "vpmc_transport.cuh"

namespace vpk {

// history id <-> work item (C2)
struct WorkMap {
    int mode;                         // 0 dose, 1 influence
    unsigned long long n_items;       // items of this launch
    unsigned long long item0;         // first item of this launch within the batch
    const unsigned long long *cum;    // dose: [n_spots+1] prefix of this batch's per-spot item counts
    const unsigned long long *first;  // dose: [n_spots] first history id of this batch's sub-range of spot j
    int n_spots;
    unsigned int hps;                 // influence: histories per spot
    int g0;                           // influence: first global spot (column) of this launch
};

// survivors of the beam line, SoA of 16-byte records for coalesced access
struct Queue {
    float4 *q0;   // lx, ly, lz (local offsets in the entry voxel), E
    float4 *q1;   // ux, uy, uz, t_rad    (CT frame)
    float4 *q2;   // tau, tau_star, step (bits), R low word
    uint4 *q3;    // hid_lo, hid_hi, voxel linear index, R high word
    unsigned int *count;   // entries pushed
    unsigned int *head;    // entries claimed by the voxel kernel
    unsigned int capacity;
};

// influence-mode scoring target (S7): per-column private box in CT index space + overflow list
struct ColumnBoxes {
    const int4 *lo;          // [n_cols] box low corner (ix, iy, iz, 0)
    const int4 *dim;         // [n_cols] box extent (bx, by, bz, 0)
    const unsigned long long *offset;   // [n_cols] offset of the box in `scratch`
    float *scratch;          // concatenated boxes
    unsigned int *ovf_count; // overflow entries appended
    unsigned int ovf_capacity;
    int *ovf_col; int *ovf_vox; float *ovf_val;
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
__device__ __forceinline__ unsigned warp_sum(unsigned v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// block-level reduction of the per-thread tallies, then 13 global atomics per block
__device__ void flush_tallies(const Tally &t, DevTallies *g)
{
    __shared__ double sd[6];
    __shared__ unsigned int sc[7];
    if (threadIdx.x < 6) sd[threadIdx.x] = 0.0;
    if (threadIdx.x < 7) sc[threadIdx.x] = 0u;
    __syncthreads();
    const double d[6] = { t.incident, t.dep_ct, t.dep_rs, t.dep_brass, t.escaped, t.removed };
    const unsigned c[7] = { t.n_stopped_ct, t.n_stopped_rs, t.n_stopped_brass, t.n_nuclear, t.n_escaped, t.n_steps_ct, t.n_steps_dev };
    const int lane = threadIdx.x & 31;
#pragma unroll
    for (int i = 0; i < 6; ++i) { const double v = warp_sum(d[i]); if (lane == 0 && v != 0.0) atomicAdd(&sd[i], v); }
#pragma unroll
    for (int i = 0; i < 7; ++i) { const unsigned v = warp_sum(c[i]); if (lane == 0 && v) atomicAdd(&sc[i], v); }
    __syncthreads();
    if (threadIdx.x < 6 && sd[threadIdx.x] != 0.0) atomicAdd(&g->incident + threadIdx.x, sd[threadIdx.x]);
    if (threadIdx.x < 7 && sc[threadIdx.x]) atomicAdd(&g->n_stopped_ct + threadIdx.x, (unsigned long long)sc[threadIdx.x]);
}

// item -> (global spot, history id)
__device__ __forceinline__ void map_item(const WorkMap &wm, unsigned long long k, int &g, unsigned long long &hid)
{
    if (wm.mode == 0) {
        int lo = 0, hi = wm.n_spots;           // largest g with cum[g] <= k and a non-empty range
        while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (__ldg(wm.cum + mid) <= k) lo = mid; else hi = mid; }
        g = lo;
        hid = __ldg(wm.first + g) + (k - __ldg(wm.cum + g));
    } else {
        const unsigned long long c = k / wm.hps;
        g = wm.g0 + (int)c;
        hid = (unsigned long long)g * wm.hps + (k - c * wm.hps);
    }
}

// ------------------------------------------------------------------------------------------- S1-S3
__global__ void __launch_bounds__(256)
beamline_kernel(const DevParams P, const DevGrid G, const WorkMap wm, const float4 *__restrict__ spots,
                const double *__restrict__ spot_R0, const int *__restrict__ spot_beam, const DevBeam *__restrict__ beams, const float3 shift,
                const uint32_t k0, const uint32_t k1, const Queue q, DevTallies *tal)
{
    const unsigned long long k = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    Tally t;
    Hist h;
    int iv[3] = { 0, 0, 0 };
    int g = 0;
    bool alive = false;
    if (k < wm.n_items) {
        unsigned long long hid;
        map_item(wm, wm.item0 + k, g, hid);
        h.hid_lo = (uint32_t)hid; h.hid_hi = (uint32_t)(hid >> 32);
        const DevBeam b = beams[__ldg(spot_beam + g)];
        sample_source(P, __ldg(spots + g), __ldg(spot_R0 + g), h, k0, k1);
        t.incident = (double)h.E;
        NullTracer tr;
        const float sh[3] = { shift.x, shift.y, shift.z };
        float w_now;
        if (beamline(P, b, h, t, tr, k0, k1, w_now) == CONT) alive = enter_ct(G, b, sh, w_now, h, iv, t, tr) == CONT;
        t.n_steps_dev = h.step;
    }
    // S6b, first stage: only survivors enter the voxel queue (warp-aggregated slot claim)
    const unsigned mask = __ballot_sync(0xffffffffu, alive);
    if (mask) {
        unsigned base = 0;
        const int leader = __ffs(mask) - 1;
        if ((threadIdx.x & 31) == leader) base = atomicAdd(q.count, __popc(mask));
        base = __shfl_sync(0xffffffffu, base, leader);
        if (alive) {
            const unsigned slot = base + __popc(mask & lanemask_lt());
            if (slot < q.capacity) {
                q.q0[slot] = make_float4(h.rx, h.ry, h.rz, h.E);
                q.q1[slot] = make_float4(h.ux, h.uy, h.uz, h.t_rad);
                const unsigned long long rb = (unsigned long long)__double_as_longlong(h.R);
                q.q2[slot] = make_float4(h.tau, h.tau_star, __uint_as_float(h.step), __uint_as_float((unsigned)rb));
                q.q3[slot] = make_uint4(h.hid_lo, h.hid_hi, (unsigned)(iv[0] + G.nx * (iv[1] + G.ny * iv[2])), (unsigned)(rb >> 32));
            }
        }
    }
    flush_tallies(t, tal);
}

// ------------------------------------------------------------------------------------------- S4-S6
// One CT step of history h in voxel (ix,iy,iz): returns the cause; v = voxel of the deposit, o.dep its size.
template <class Tracer, class Lut>
__device__ __forceinline__ int ct_step(const DevParams &P, const DevGrid &G, const short *__restrict__ hu, const Lut &lut,
                                       float rsp_scale, Hist &h, int &ix, int &iy, int &iz, long long &v, StepOut &o,
                                       Tracer &tr, uint32_t k0, uint32_t k1)
{
    int ax;
    const float d = face_distance(G, h, ax);
    const bool up = (ax == 0 ? h.ux : (ax == 1 ? h.uy : h.uz)) > 0.0f;   // direction of travel during the step
    v = ix + (long long)G.nx * (iy + (long long)G.ny * iz);
    int t = (int)__ldg(hu + v) - G.hu_min;
    t = min(max(t, 0), G.n_lut - 1);
    const float4 mv = lut[t];
    const Medium m = { mv.x * rsp_scale, mv.y, mv.z, mv.w };
    const float Eb = h.E; const uint32_t st = h.step;
    const int iv0[3] = { ix, iy, iz };
    int cause = material_step(P, h, m, d, k0, k1, o);
    if (cause == CONT && o.on_d && cross_face(G, h, ix, iy, iz, ax, up)) cause = ESCAPED;
    tr.put(h, fmaf((float)ix, G.hx, G.ox), fmaf((float)iy, G.hy, G.oy), fmaf((float)iz, G.hz, G.oz), st, REG_CT, iv0,
           Eb, h.E, o.s, cause);
    return cause;
}

struct LutShared { const float4 *p; __device__ __forceinline__ float4 operator[](int i) const { return p[i]; } };
struct LutGlobal { const float4 *p; __device__ __forceinline__ float4 operator[](int i) const { return __ldg(p + i); } };

// MODE 0: dose grid; MODE 1: per-column boxes.  SMEM_LUT: material table staged in shared memory.
template <int MODE, bool SMEM_LUT>
__global__ void __launch_bounds__(256)
voxel_kernel(const DevParams P, const DevGrid G, const Queue q, const short *__restrict__ hu,
             const float4 *__restrict__ lut_g, const float rsp_scale, float *__restrict__ edep,
             const ColumnBoxes cb, const int col0, const unsigned int hps, const uint32_t k0, const uint32_t k1,
             DevTallies *tal)
{
    extern __shared__ float4 lut_s[];
    if (SMEM_LUT) {
        for (int i = threadIdx.x; i < G.n_lut; i += blockDim.x) lut_s[i] = lut_g[i];
        __syncthreads();
    }
    const unsigned n_q = min(*q.count, q.capacity);
    const int lane = threadIdx.x & 31;
    Tally t;
    Hist h;
    int ix = 0, iy = 0, iz = 0, col = 0;
    float hdep = 0.0f;
    bool alive = false, exhausted = false;
    NullTracer tr;
    for (;;) {
        // S6b: refill dead lanes from the queue (one atomic per warp)
        const unsigned need = __ballot_sync(0xffffffffu, !alive);
        if (need && !exhausted) {
            unsigned base = 0;
            const int leader = __ffs(need) - 1;
            const int cnt = __popc(need);
            if (lane == leader) base = atomicAdd(q.head, cnt);
            base = __shfl_sync(0xffffffffu, base, leader);
            exhausted = base + cnt >= n_q;
            if (!alive) {
                const unsigned slot = base + __popc(need & lanemask_lt());
                if (slot < n_q) {
                    const float4 a = q.q0[slot], b = q.q1[slot], c = q.q2[slot];
                    const uint4 e = q.q3[slot];
                    h.rx = a.x; h.ry = a.y; h.rz = a.z; h.E = a.w;
                    h.ux = b.x; h.uy = b.y; h.uz = b.z; h.t_rad = b.w; h.A_rad = highland_A(b.w, P.c_log);
                    h.tau = c.x; h.tau_star = c.y; h.step = __float_as_uint(c.z);
                    h.R = __longlong_as_double((long long)(((unsigned long long)e.w << 32) | __float_as_uint(c.w)));
                    h.hid_lo = e.x; h.hid_hi = e.y;
                    iz = (int)(e.z / (unsigned)(G.nx * G.ny));
                    const int rem = (int)(e.z - (unsigned)iz * (unsigned)(G.nx * G.ny));
                    iy = rem / G.nx; ix = rem - iy * G.nx;
                    if (MODE == 1) col = (int)((((unsigned long long)e.y << 32) | e.x) / hps);
                    hdep = 0.0f;
                    alive = true;
                }
            }
        }
        if (!__any_sync(0xffffffffu, alive)) break;
        if (alive) {
            long long v; StepOut o;
            int cause;
            const int vx = ix, vy = iy, vz = iz;      // voxel of the deposit = voxel at the start of the step
            if (SMEM_LUT) cause = ct_step(P, G, hu, LutShared{ lut_s }, rsp_scale, h, ix, iy, iz, v, o, tr, k0, k1);
            else cause = ct_step(P, G, hu, LutGlobal{ lut_g }, rsp_scale, h, ix, iy, iz, v, o, tr, k0, k1);
            t.n_steps_ct += (cause != STOPPED);
            if (o.dep != 0.0f) {
                if (MODE == 0) {
                    atomicAdd(edep + v, o.dep);
                } else {
                    const int c = col - col0;
                    const int4 lo = __ldg(cb.lo + c), dm = __ldg(cb.dim + c);
                    const int bx = vx - lo.x, by = vy - lo.y, bz = vz - lo.z;
                    if ((unsigned)bx < (unsigned)dm.x && (unsigned)by < (unsigned)dm.y && (unsigned)bz < (unsigned)dm.z) {
                        atomicAdd(cb.scratch + __ldg(cb.offset + c) + (bx + (unsigned long long)dm.x * (by + (unsigned long long)dm.y * bz)), o.dep);
                    } else {
                        const unsigned s = atomicAdd(cb.ovf_count, 1u);
                        if (s < cb.ovf_capacity) { cb.ovf_col[s] = col; cb.ovf_vox[s] = (int)v; cb.ovf_val[s] = o.dep; }
                    }
                }
                hdep += o.dep;
            }
            if (cause != CONT) {
                t.dep_ct += (double)hdep;
                t.removed += (double)o.removed;
                book_end(t, cause, REG_CT, cause == ESCAPED ? h.E : 0.0f);
                alive = false;
            }
        }
    }
    flush_tallies(t, tal);
}

// ------------------------------------------------------------------------------------------- trace
template <bool DUMMY>
__global__ void trace_kernel(const DevParams P, const DevGrid G, const unsigned long long *__restrict__ hids,
                             const int *__restrict__ spot_of, int n, const float4 *__restrict__ spots,
                             const double *__restrict__ spot_R0, const int *__restrict__ spot_beam, const DevBeam *__restrict__ beams, const float3 shift,
                             const short *__restrict__ hu, const float4 *__restrict__ lut_g, float rsp_scale,
                             uint32_t k0, uint32_t k1, StepRec *recs, int max_steps, int *nrec)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    RecTracer tr{ recs + (size_t)i * max_steps, max_steps, 0 };
    const int g = spot_of[i];
    if (g < 0) { nrec[i] = 0; return; }
    Hist h; Tally t;
    h.hid_lo = (uint32_t)hids[i]; h.hid_hi = (uint32_t)(hids[i] >> 32);
    const DevBeam b = beams[spot_beam[g]];
    sample_source(P, spots[g], spot_R0[g], h, k0, k1);
    int iv[3];
    const float sh[3] = { shift.x, shift.y, shift.z };
    float w_now;
    if (beamline(P, b, h, t, tr, k0, k1, w_now) == CONT && enter_ct(G, b, sh, w_now, h, iv, t, tr) == CONT) {
        int ix = iv[0], iy = iv[1], iz = iv[2];
        for (int it = 0; it < 1000000; ++it) {
            long long v; StepOut o;
            if (ct_step(P, G, hu, LutGlobal{ lut_g }, rsp_scale, h, ix, iy, iz, v, o, tr, k0, k1) != CONT) break;
        }
    }
    nrec[i] = tr.n;
}

// ------------------------------------------------------------------------------------------- S6 / C6
// fold one batch into the running sums; f = N / N_b scales the batch to full weight
__global__ void batch_accumulate_kernel(float *__restrict__ edep_b, float *__restrict__ sum, float *__restrict__ s1,
                                        float *__restrict__ s2, long long n, float f, int with_unc)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x; v < n; v += stride) {
        const float x = edep_b[v];
        if (x != 0.0f) {
            edep_b[v] = 0.0f;
            sum[v] += x;
            if (with_unc) { const float y = f * x; s1[v] += y; s2[v] = fmaf(y, y, s2[v]); }
        }
    }
}

// dose[v] = scale * E_dep[v] / (max(rho_v, rho_min) V[cm3]) * 1.602176634e-10 Gy
__global__ void dose_convert_kernel(const float *__restrict__ sum, const short *__restrict__ hu,
                                    const float4 *__restrict__ lut, DevGrid G, float rho_min, float coef,
                                    float *__restrict__ dose, long long n, unsigned int *max_bits)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    float mx = 0.0f;
    for (long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x; v < n; v += stride) {
        int t = (int)__ldg(hu + v) - G.hu_min;
        t = min(max(t, 0), G.n_lut - 1);
        const float rho = fmaxf(__ldg(lut + t).y, rho_min);
        const float dv = __fdiv_rn(coef * sum[v], rho);
        dose[v] = dv;
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

}  // namespace vpk
