// vpmc_gamma.cuh -- SURVEY.md 8(f)-3, second half: the 3-D gamma index ("3D Gamma passing rate"; Low et al., ref. 80) as
// kernels, so a dose comparison needs no host pass over the grids.  S:8c-C6: global normalisation to the reference maximum,
// voxels with reference dose >= threshold x maximum are evaluated, gamma <= 1 passes; the zero-distance test first, the full
// search (evaluated dose interpolated trilinearly on a lattice of h / sub inside the distance-to-agreement sphere, edge
// values beyond the grid) only for the voxels that fail it.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace vpk {

struct GammaArgs {
    int nx, ny, nz;
    float hx, hy, hz;
    float dd_rel, dta, thr_rel;
    int sub;
};

struct GammaCounts { unsigned long long n_eval, n_zero_fail, n_fail; unsigned int max_bits, pad_; };

__global__ void gamma_max_kernel(const float *__restrict__ ref, long long n, GammaCounts *c)
{
    float mx = 0.0f;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x; v < n; v += stride) mx = fmaxf(mx, ref[v]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    if ((threadIdx.x & 31) == 0 && mx > 0.0f) atomicMax(&c->max_bits, __float_as_uint(mx));
}

// zero-distance test; the voxels that fail it are listed for the search
__global__ void gamma_select_kernel(const float *__restrict__ ref, const float *__restrict__ ev, long long n, GammaArgs a, GammaCounts *c,
                                    unsigned int *__restrict__ list, unsigned int cap)
{
    const float mx = __uint_as_float(c->max_bits);
    const float dcrit = a.dd_rel * mx, lo = a.thr_rel * mx;
    const long long stride = (long long)gridDim.x * blockDim.x;
    unsigned int n_eval = 0;
    for (long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x; v < n; v += stride) {
        const float r = ref[v];
        if (!(r >= lo)) continue;
        n_eval += 1u;
        if (fabsf(ev[v] - r) > dcrit) {
            const unsigned long long slot = atomicAdd(&c->n_zero_fail, 1ull);
            if (slot < cap) list[slot] = (unsigned int)v;
        }
    }
    n_eval = __reduce_add_sync(0xffffffffu, n_eval);
    if ((threadIdx.x & 31) == 0 && n_eval) atomicAdd(&c->n_eval, (unsigned long long)n_eval);
}

__device__ __forceinline__ float gamma_fetch(const float *__restrict__ ev, const GammaArgs &a, int x, int y, int z)
{
    x = min(max(x, 0), a.nx - 1); y = min(max(y, 0), a.ny - 1); z = min(max(z, 0), a.nz - 1);
    return __ldg(ev + x + (size_t)a.nx * (y + (size_t)a.ny * z));
}

// one warp per listed voxel: the lanes share the lattice points of the search sphere; the voxel passes as soon as any lane
// finds gamma^2 <= 1
__global__ void __launch_bounds__(256)
gamma_search_kernel(const float *__restrict__ ref, const float *__restrict__ ev, GammaArgs a, GammaCounts *c, const unsigned int *__restrict__ list,
                    unsigned int cap)
{
    const unsigned int n_list = (unsigned int)min((unsigned long long)cap, c->n_zero_fail);
    const int lane = threadIdx.x & 31;
    const unsigned int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, n_warps = (gridDim.x * blockDim.x) >> 5;
    const float mx = __uint_as_float(c->max_bits);
    const float inv_dcrit = 1.0f / (a.dd_rel * mx), inv_sub = 1.0f / (float)a.sub, inv_dta2 = 1.0f / (a.dta * a.dta);
    const int kx = (int)ceilf(a.dta / a.hx * (float)a.sub), ky = (int)ceilf(a.dta / a.hy * (float)a.sub), kz = (int)ceilf(a.dta / a.hz * (float)a.sub);
    const int wx = 2 * kx + 1, wy = 2 * ky + 1, wz = 2 * kz + 1;
    const int n_pts = wx * wy * wz;
    unsigned int fails = 0;
    for (unsigned int i = warp; i < n_list; i += n_warps) {
        const unsigned int v = list[i];
        const int z = (int)(v / (unsigned)(a.nx * a.ny)), rem = (int)(v - (unsigned)z * (unsigned)(a.nx * a.ny)), y = rem / a.nx, x = rem - y * a.nx;
        const float r = __ldg(ref + v);
        bool pass = false;
        for (int p0 = 0; p0 < n_pts && !pass; p0 += 32) {
            const int p = p0 + lane;
            bool ok = false;
            if (p < n_pts) {
                const int iz = p / (wx * wy), q = p - iz * wx * wy, iy = q / wx, ix = q - iy * wx;
                const float ox = (float)(ix - kx) * inv_sub, oy = (float)(iy - ky) * inv_sub, oz = (float)(iz - kz) * inv_sub;      // voxel units
                const float d2 = ((ox * a.hx) * (ox * a.hx) + (oy * a.hy) * (oy * a.hy) + (oz * a.hz) * (oz * a.hz)) * inv_dta2;
                if (d2 <= 1.0f) {
                    const float fx = floorf(ox), fy = floorf(oy), fz = floorf(oz);
                    const float tx = ox - fx, ty = oy - fy, tz = oz - fz;
                    const int x0 = x + (int)fx, y0 = y + (int)fy, z0 = z + (int)fz;
                    const float c00 = gamma_fetch(ev, a, x0, y0, z0) * (1.0f - tx) + gamma_fetch(ev, a, x0 + 1, y0, z0) * tx;
                    const float c10 = gamma_fetch(ev, a, x0, y0 + 1, z0) * (1.0f - tx) + gamma_fetch(ev, a, x0 + 1, y0 + 1, z0) * tx;
                    const float c01 = gamma_fetch(ev, a, x0, y0, z0 + 1) * (1.0f - tx) + gamma_fetch(ev, a, x0 + 1, y0, z0 + 1) * tx;
                    const float c11 = gamma_fetch(ev, a, x0, y0 + 1, z0 + 1) * (1.0f - tx) + gamma_fetch(ev, a, x0 + 1, y0 + 1, z0 + 1) * tx;
                    const float val = (c00 * (1.0f - ty) + c10 * ty) * (1.0f - tz) + (c01 * (1.0f - ty) + c11 * ty) * tz;
                    const float e = (val - r) * inv_dcrit;
                    ok = d2 + e * e <= 1.0f;
                }
            }
            pass = __any_sync(0xffffffffu, ok);
        }
        fails += pass ? 0u : 1u;
    }
    if (lane == 0 && fails) atomicAdd(&c->n_fail, (unsigned long long)fails);
}

}  // namespace vpk
