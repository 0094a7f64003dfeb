// vpmc_spmv.cuh -- SURVEY.md 8(f)-1: one iteration of the robust optimiser on the CSR influence matrices the transport path
// writes ("0.1-0.3 s per iteration", P:L160 13 scenarios).  Rows = spots, columns = voxels (C6), so
//   dose  d[v] = sum_j D[j][v] w[j]   is a SCATTER over the rows   (spmv_dose_kernel: fp32 REDs, coalesced because a row's
//                                                                   entries ascend in voxel index),
//   grad  g[j] = sum_v D[j][v] r[v]   is a GATHER per row          (spmv_grad_kernel + spmv_grad_fixup_kernel, deterministic),
// and the voxel-wise worst case over the scenarios (R16) is one elementwise pass (worst_case_kernel).
// All three are HBM-bound: 8 B per stored entry (4 B column index + 4 B value) stream through once per product; the
// vectors (w: n_spots floats, r / d: one float per voxel, 42 MB for the head CT) stay in L2.
// The work is cut by ENTRIES, not by rows: CTA b owns entries [b kSpmvChunk, (b+1) kSpmvChunk), so the load is balanced
// whatever the row lengths (5 10^4 entries per row in config 4, but also empty rows).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace vpk {

constexpr int kSpmvBlock = 256;
constexpr int kSpmvChunk = 8192;          // entries per CTA

// row of entry k: the j with row_ptr[j] <= k < row_ptr[j + 1], searched in [lo, hi) (invariant row_ptr[lo] <= k < row_ptr[hi])
__device__ __forceinline__ int spmv_row_of(const long long *__restrict__ row_ptr, int lo, int hi, long long k)
{
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (__ldg(row_ptr + mid) <= k) lo = mid; else hi = mid;
    }
    return lo;
}

__device__ __forceinline__ void spmv_chunk_rows(const long long *__restrict__ row_ptr, int n_rows, long long base, long long end, int &j0, int &j1)
{
    __shared__ int s_j[2];
    if (threadIdx.x == 0) s_j[0] = spmv_row_of(row_ptr, 0, n_rows, base);
    if (threadIdx.x == 32) s_j[1] = spmv_row_of(row_ptr, 0, n_rows, end - 1);
    __syncthreads();
    j0 = s_j[0]; j1 = s_j[1];
}

// d[col[k]] += val[k] * w[row(k)] for the CTA's entries; d zeroed beforehand.  One lane per entry: a warp's 32 entries are
// (mostly) 32 consecutive voxels, i.e. four 32-byte sectors per RED instruction.
__global__ void __launch_bounds__(kSpmvBlock)
spmv_dose_kernel(const long long *__restrict__ row_ptr, const int *__restrict__ col, const float *__restrict__ val, int n_rows,
                 long long nnz, const float *__restrict__ w, float *__restrict__ d)
{
    const long long base = (long long)blockIdx.x * kSpmvChunk, end = min(base + (long long)kSpmvChunk, nnz);
    int j0, j1;
    spmv_chunk_rows(row_ptr, n_rows, base, end, j0, j1);
    const float w0 = __ldg(w + j0);
    const long long e0 = __ldg(row_ptr + j0 + 1);          // end of the first row
#pragma unroll 4
    for (long long k = base + threadIdx.x; k < end; k += kSpmvBlock) {
        const int c = __ldg(col + k);
        const float x = __ldg(val + k);
        const float wj = (k < e0) ? w0 : __ldg(w + spmv_row_of(row_ptr, j0, j1 + 1, k));
        atomicAdd(d + c, x * wj);
    }
}

// block sum in a fixed order (warp shuffles, then the warps' sums in warp order)
__device__ __forceinline__ float spmv_block_sum(float v, float *s_w)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    __syncthreads();                                        // s_w may still be read from the previous call
    if ((threadIdx.x & 31) == 0) s_w[threadIdx.x >> 5] = v;
    __syncthreads();
    float t = 0.0f;
#pragma unroll
    for (int i = 0; i < kSpmvBlock / 32; ++i) t += s_w[i];
    return t;
}

// Per CTA, for every row that has entries in the CTA's range: the partial sum of val * r[col] over that part of the row.
// A row that lies entirely inside the range is finished here (g[j] written); of the others there are at most two per CTA --
// the row that holds the CTA's first entry (-> first_part[b]) and a row that starts inside and runs beyond the end
// (-> last_part[b]) -- and spmv_grad_fixup_kernel adds their parts in chunk order: the result does not depend on timing.
__global__ void __launch_bounds__(kSpmvBlock)
spmv_grad_kernel(const long long *__restrict__ row_ptr, const int *__restrict__ col, const float *__restrict__ val, int n_rows,
                 long long nnz, const float *__restrict__ r, float *__restrict__ g, int accumulate, float *__restrict__ first_part,
                 float *__restrict__ last_part)
{
    __shared__ float s_w[kSpmvBlock / 32];
    const long long base = (long long)blockIdx.x * kSpmvChunk, end = min(base + (long long)kSpmvChunk, nnz);
    int j0, j1;
    spmv_chunk_rows(row_ptr, n_rows, base, end, j0, j1);
    for (int j = j0; j <= j1; ++j) {
        const long long ra = __ldg(row_ptr + j), rb = __ldg(row_ptr + j + 1);
        if (ra == rb) continue;                             // empty row inside the range
        const long long a = max(ra, base), b = min(rb, end);
        float acc[4] = { 0.0f, 0.0f, 0.0f, 0.0f };
        long long k = a + threadIdx.x;
        for (; k + 3 * kSpmvBlock < b; k += 4 * kSpmvBlock) {
#pragma unroll
            for (int u = 0; u < 4; ++u) acc[u] = fmaf(__ldg(val + k + u * kSpmvBlock), __ldg(r + __ldg(col + k + u * kSpmvBlock)), acc[u]);
        }
        for (; k < b; k += kSpmvBlock) acc[0] = fmaf(__ldg(val + k), __ldg(r + __ldg(col + k)), acc[0]);
        const float s = spmv_block_sum((acc[0] + acc[1]) + (acc[2] + acc[3]), s_w);
        if (threadIdx.x == 0) {
            if (ra >= base && rb <= end) g[j] = accumulate ? g[j] + s : s;
            else if (ra <= base) first_part[blockIdx.x] = s;
            else last_part[blockIdx.x] = s;
        }
    }
}

// rows that span several chunks (their parts added in chunk order) and empty rows
__global__ void spmv_grad_fixup_kernel(const long long *__restrict__ row_ptr, int n_rows, const float *__restrict__ first_part,
                                       const float *__restrict__ last_part, float *__restrict__ g, int accumulate)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_rows) return;
    const long long a = __ldg(row_ptr + j), b = __ldg(row_ptr + j + 1);
    if (a == b) { if (!accumulate) g[j] = 0.0f; return; }
    const long long c0 = a / kSpmvChunk, c1 = (b - 1) / kSpmvChunk;
    if (c0 == c1) return;                                   // finished by spmv_grad_kernel
    float s = 0.0f;
    for (long long c = c0; c <= c1; ++c) s += (c == c0 && a > c0 * kSpmvChunk) ? last_part[c] : first_part[c];
    g[j] = accumulate ? g[j] + s : s;
}

// DESIGN.md R16: per voxel the scenario with the largest squared deviation from the target (lowest index among equals);
// resid_s[v] = 2 p[v] (d_s[v] - t[v]) for that scenario, 0 for the others; objective += sum_v p[v] e^2 (fp64).
__global__ void __launch_bounds__(256)
worst_case_kernel(const float *__restrict__ doses, int n_sc, long long n, const float *__restrict__ target, const float *__restrict__ weight,
                  float *__restrict__ resid, double *__restrict__ objective)
{
    double f = 0.0;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x; v < n; v += stride) {
        const float t = __ldg(target + v), p = __ldg(weight + v);
        int best = 0;
        float e_best = __fsub_rn(doses[v], t);
        float q_best = __fmul_rn(e_best, e_best);
        for (int s = 1; s < n_sc; ++s) {
            const float e = __fsub_rn(doses[(size_t)s * n + v], t);
            const float q = __fmul_rn(e, e);
            if (q > q_best) { e_best = e; best = s; q_best = q; }
        }
        for (int s = 0; s < n_sc; ++s) resid[(size_t)s * n + v] = (s == best) ? 2.0f * p * e_best : 0.0f;
        f += (double)p * (double)e_best * (double)e_best;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) f += __shfl_xor_sync(0xffffffffu, f, o);
    if ((threadIdx.x & 31) == 0 && f != 0.0) atomicAdd(objective, f);
}

}  // namespace vpk
