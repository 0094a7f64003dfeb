// vpmc_setup.cuh -- S0 on the device: the per-aperture tables (packed opening bitmap, the two safe-distance maps of
// DESIGN.md 5.2) are built from the caller's uint8 bitmap by kernels on the handle's set-up stream, so a plan's set-up costs
// one host->device copy and a handful of launches instead of host loops over 10^5-10^6 pixels; and the measurement kernel of
// SURVEY.md 8(d)(iii) (random fp32 RED into an L2-resident buffer).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "vpmc_device.cuh"

namespace vpk {

// packed bitmap: bit (ix & 31) of word ix >> 5 of row iy; one thread per padded pixel, one ballot per word
__global__ void ap_pack_kernel(const unsigned char *__restrict__ open, int nx, int ny, int rw, uint32_t *__restrict__ bits)
{
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int wpr = rw * 32;
    const int iy = (int)(idx / wpr), ix = (int)(idx - (long long)iy * wpr);
    const bool o = iy < ny && ix < nx && open[(size_t)iy * nx + ix] != 0;
    const unsigned m = __ballot_sync(0xffffffffu, o);
    if ((threadIdx.x & 31) == 0 && iy < ny) bits[(size_t)iy * rw + (ix >> 5)] = m;
}

// per tile of 2^shift x 2^shift pixels: bit 0 = every pixel of the tile is open (and the tile lies inside the bitmap),
// bit 1 = some pixel is open
__global__ void ap_tile_flags_kernel(const unsigned char *__restrict__ open, int nx, int ny, int shift, int ntx, int nty,
                                     unsigned char *__restrict__ flags)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ntx * nty) return;
    const int ty = t / ntx, tx = t - ty * ntx, ts = 1 << shift;
    bool all = (tx + 1) * ts <= nx && (ty + 1) * ts <= ny, any = false;
    for (int iy = ty * ts; iy < min((ty + 1) * ts, ny); ++iy)
        for (int ix = tx * ts; ix < min((tx + 1) * ts, nx); ++ix) {
            const bool o = open[(size_t)iy * nx + ix] != 0;
            all = all && o; any = any || o;
        }
    flags[t] = (unsigned char)((all ? 1 : 0) | (any ? 2 : 0));
}

// Chebyshev distance maps, capped at 255, exact: D(x, y) = min over sources (x', y') of max(|x - x'|, |y - y'|)
//   = min over k of max(k, min(c(x - k, y), c(x + k, y))),  c(x, y) = distance along the column x to its nearest source.
// Map 0 ("to brass"): sources = tiles that are not fully open, and everything outside the bitmap.
// Map 1 ("to the opening"): sources = tiles with any open pixel; nothing outside.
// Pass 1, one thread per column: c for both maps (two sweeps, coalesced across the threads of a warp).
__global__ void ap_dist_columns_kernel(const unsigned char *__restrict__ flags, int ntx, int nty, unsigned char *__restrict__ c_br,
                                       unsigned char *__restrict__ c_op)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= ntx) return;
    int db = 0, dp = 255;                 // above row 0: brass (a source of map 0), no opening
    for (int y = 0; y < nty; ++y) {
        const unsigned char f = flags[(size_t)y * ntx + x];
        db = (f & 1) ? min(db + 1, 255) : 0;
        dp = (f & 2) ? 0 : min(dp + 1, 255);
        c_br[(size_t)y * ntx + x] = (unsigned char)db; c_op[(size_t)y * ntx + x] = (unsigned char)dp;
    }
    db = 0; dp = 255;
    for (int y = nty - 1; y >= 0; --y) {
        const unsigned char f = flags[(size_t)y * ntx + x];
        db = (f & 1) ? min(db + 1, 255) : 0;
        dp = (f & 2) ? 0 : min(dp + 1, 255);
        const size_t i = (size_t)y * ntx + x;
        c_br[i] = (unsigned char)min((int)c_br[i], db); c_op[i] = (unsigned char)min((int)c_op[i], dp);
    }
}

// Pass 2, one thread per tile and map: the search over k stops as soon as k reaches the best value found
__global__ void ap_dist_rows_kernel(const unsigned char *__restrict__ c_br, const unsigned char *__restrict__ c_op, int ntx, int nty,
                                    unsigned char *__restrict__ dist /* [2][nty][ntx] */)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const int n = ntx * nty;
    if (t >= 2 * n) return;
    const int map = t / n, r = t - map * n, y = r / ntx, x = r - y * ntx;
    const unsigned char *c = (map ? c_op : c_br) + (size_t)y * ntx;
    int best = c[x];
    for (int k = 1; k < best; ++k) {
        int v = 255;
        if (x - k >= 0) v = c[x - k]; else if (map == 0) v = 0;       // left of the bitmap: brass
        if (x + k < ntx) v = min(v, (int)c[x + k]); else if (map == 0) v = 0;
        best = min(best, max(k, v));
    }
    dist[t] = (unsigned char)best;
}

// ceiling of global fp32 RED throughput -- every thread adds to pseudo-random elements of a buffer
// that stays L2-resident (the addresses come from a 32-bit LCG, so address generation is two integer instructions per RED)
__global__ void red_ceiling_kernel(float *__restrict__ buf, unsigned int mask, unsigned int per_thread)
{
    unsigned int s = (blockIdx.x * blockDim.x + threadIdx.x) * 2654435761u + 12345u;
#pragma unroll 4
    for (unsigned int i = 0; i < per_thread; ++i) {
        s = s * 1664525u + 1013904223u;
        atomicAdd(buf + ((s >> 8) & mask), 1.0f);
    }
}

}  // namespace vpk
