// rt_ray_sort.cuh — the thread -> ray map of marches over grids far larger than the L2 (sm_100a): the rays of ALL
// sources sorted by the tile of the grid they are in half-way along the marched path and, within a tile, by direction,
// so that the blocks in flight load and reduce into one neighbourhood of the grid instead of all of it.
//
// Eq. (2) fixes the order of the substeps of ONE ray only; rays are independent, so any
// assignment of rays to threads gives the same sums.  With few sources in a large grid (C4: 64 sources, 16,384 rays
// each, 256^3 x 4 bins) neither of the static maps of rt_common.cuh keeps the traffic local: a warp of 32 sources x one
// direction touches 32 distant places, and blocks of one source's directions fan out over the whole grid; ncu showed
// the march moving 54.6 GB through HBM in 32-byte sectors (20 x the grids it reads and writes).  Rays that are in
// the same tile at the same substep and travel the same way -- from whatever source -- march next to each other
// instead, and stay next to each other for most of their path (C4 26.2 -> 13.9 ms).
// KEY = Morton code of the 32^3-cell tile at mid-path (coarser on grids beyond 512 cells per axis: at most 16 tiles per
// axis), then 7 bits of direction: the face of the cube map the direction points through and the cell of a 4 x 4 grid on
// that face.  Measured on C4 (ms per call): 8^3 tiles alone 14.8, 16^3 + octant 14.2, 16^3 + 4 x 4 per face 14.1,
// 32^3 + 4 x 4 13.9 (8 x 8: 13.9), 64^3 + 4 x 4 14.6, 128^3 + 8 x 8 16.7, direction only 19.8.
// The sort is a locality heuristic: keys are computed in double, not in the march's fixed point, and the order of rays
// with equal keys is whatever the scatter's atomics give -- neither changes a deposit.
#pragma once
#include "rt_common.cuh"

namespace rt {

constexpr int kRayDirBits = 7;                      // 6 faces x 4 x 4 cells = 96 direction bins
constexpr int kRayTiles = 1 << (12 + kRayDirBits);  // the largest key space: 16^3 tiles x 128 (the workspace holds this many)

// a tile is (1 << shift)^3 cells -- 32^3, or larger so that an axis has at most 16 tiles -- and the tile index of an axis
// takes `bits` bits; n_keys = the key space in use, a multiple of 4096
struct RaySortGeom {
    int shift, bits, n_keys;
};
__host__ __device__ inline RaySortGeom ray_sort_geom(int nx, int ny, int nz) {
    int m = nx > ny ? nx : ny;
    m = m > nz ? m : nz;
    RaySortGeom g;
    g.shift = 5;
    while (((m - 1) >> g.shift) >= 16) ++g.shift;
    g.bits = 1;
    while (((m - 1) >> g.shift) >= (1 << g.bits)) ++g.bits;
    const int n = (1 << (3 * g.bits)) << kRayDirBits;
    g.n_keys = n < 4096 ? 4096 : n;
    return g;
}

__device__ __forceinline__ uint32_t spread5(uint32_t v) {      // 5 bits -> every third bit
    return (v & 1u) | ((v & 2u) << 2) | ((v & 4u) << 4) | ((v & 8u) << 6) | ((v & 16u) << 8);
}

// key[e] of ray e = source * n_rays + i: the tile it is in at substep k_mid (clamped to the grid, as its deposits are,
// PAPER.md:29) and its direction bin; hist[key]++
__global__ void ray_tile_key_kernel(uint32_t* key, uint32_t* hist, const float* sources, long long n, int n_rays, double ds,
                                    long long k_mid, int nx, int ny, int nz, RaySortGeom g) {
    const long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (e >= n) return;
    const int s = int(e / n_rays);
    const uint32_t i = uint32_t(e - (long long)s * n_rays);
    double nh[3];
    fib_direction(i, uint32_t(n_rays), nh);
    const double far = double(k_mid) * ds;
    uint32_t t[3];
    const int lim[3] = {nx - 1, ny - 1, nz - 1};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double x = double(__ldg(sources + 3 * size_t(s) + a)) + far * nh[a];
        const double c = fmin(fmax(floor(x), 0.0), double(lim[a]));       // NaN -> 0
        t[a] = uint32_t(int(c)) >> g.shift;
    }
    const uint32_t tile = (spread5(t[0]) << 2) | (spread5(t[1]) << 1) | spread5(t[2]);
    // direction: the axis of largest |n| and its sign (cube-map face), the other two components over it in [-1, 1]
    const double ax = fabs(nh[0]), ay = fabs(nh[1]), az = fabs(nh[2]);
    const int m = (ax >= ay && ax >= az) ? 0 : (ay >= az ? 1 : 2);
    const double inv = 1.0 / fmax(fabs(nh[m]), 1e-300);
    const double u = nh[(m + 1) % 3] * inv, v = nh[(m + 2) % 3] * inv;
    const int iu = min(3, max(0, int((u + 1.0) * 2.0))), iv = min(3, max(0, int((v + 1.0) * 2.0)));
    const uint32_t dir = uint32_t((2 * m + (nh[m] < 0.0 ? 1 : 0)) * 16 + iu * 4 + iv);
    const uint32_t k = ((tile << kRayDirBits) | dir) & uint32_t(g.n_keys - 1);
    key[e] = k;
    atomicAdd(hist + k, 1u);
}

// hist -> exclusive prefix sums (cursor), one block of 1024 threads, n_keys / 1024 consecutive keys per thread (a
// multiple of 4) in two passes (totals, then offsets); hist itself is zeroed for the next call
__global__ void __launch_bounds__(1024) ray_tile_scan_kernel(uint32_t* hist, uint32_t* cursor, int n_keys) {
    const int per4 = n_keys / 4096;
    __shared__ uint32_t warp_sum[32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint4* h4 = reinterpret_cast<uint4*>(hist) + size_t(threadIdx.x) * per4;
    uint32_t sum = 0;
#pragma unroll 4
    for (int i = 0; i < per4; ++i) {
        const uint4 v = h4[i];
        sum += v.x + v.y + v.z + v.w;
    }
    uint32_t incl = sum;                       // inclusive scan of the thread totals: within the warp ...
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t up = __shfl_up_sync(0xFFFFFFFFu, incl, d);
        if (lane >= d) incl += up;
    }
    if (lane == 31) warp_sum[warp] = incl;
    __syncthreads();
    if (warp == 0) {                           // ... and over the 32 warps
        uint32_t w = warp_sum[lane];
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t up = __shfl_up_sync(0xFFFFFFFFu, w, d);
            if (lane >= d) w += up;
        }
        warp_sum[lane] = w;
    }
    __syncthreads();
    uint32_t run = incl - sum + (warp ? warp_sum[warp - 1] : 0u);
    uint4* c4 = reinterpret_cast<uint4*>(cursor) + size_t(threadIdx.x) * per4;
#pragma unroll 4
    for (int i = 0; i < per4; ++i) {
        const uint4 v = h4[i];
        uint4 c;
        c.x = run; run += v.x;
        c.y = run; run += v.y;
        c.z = run; run += v.z;
        c.w = run; run += v.w;
        c4[i] = c;
        h4[i] = make_uint4(0u, 0u, 0u, 0u);
    }
}

__global__ void ray_tile_scatter_kernel(uint32_t* perm, const uint32_t* key, uint32_t* cursor, long long n) {
    const long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (e >= n) return;
    perm[atomicAdd(cursor + key[e], 1u)] = uint32_t(e);
}

}  // namespace rt
