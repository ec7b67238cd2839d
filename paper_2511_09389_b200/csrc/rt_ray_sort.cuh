// rt_ray_sort.cuh — the thread -> ray map of marches over grids far larger than the L2 (sm_100a): the rays of ALL
// sources sorted by the tile of the grid they are in half-way along the marched path, so that the blocks in flight
// load and reduce into one neighbourhood of the grid instead of all of it.
//
// Eq. (2) fixes the order of the substeps of ONE ray only; rays are independent, so any
// assignment of rays to threads gives the same sums.  With few sources in a large grid (C4: 64 sources, 16,384 rays
// each, 256^3 x 4 bins) neither of the static maps of rt_common.cuh keeps the traffic local: a warp of 32 sources x one
// direction touches 32 distant places, and blocks of one source's directions fan out over the whole grid; ncu showed
// the march moving 54.6 GB through HBM in 32-byte sectors (20 x the grids it reads and writes).  Rays that are in
// the same 8^3 tile at the same substep -- from whatever source -- march next to each other instead: C4's HBM
// traffic drops to 33 GB and the call from 26.2 to 17.3 ms.
// The sort is a locality heuristic: keys are computed in double, not in the march's fixed point, and the order of rays
// within a tile is whatever the scatter's atomics give -- neither changes a deposit.
#pragma once
#include "rt_common.cuh"

namespace rt {

constexpr int kRayTiles = 32768;      // Morton-coded tile keys: 5 bits per axis

// a tile is (1 << shift)^3 cells: 8^3, or larger so that an axis has at most 32 tiles
__host__ __device__ inline int ray_tile_shift(int nx, int ny, int nz) {
    int m = nx > ny ? nx : ny;
    m = m > nz ? m : nz;
    int shift = 3;
    while (((m - 1) >> shift) >= 32) ++shift;
    return shift;
}

__device__ __forceinline__ uint32_t spread5(uint32_t v) {      // 5 bits -> every third bit
    return (v & 1u) | ((v & 2u) << 2) | ((v & 4u) << 4) | ((v & 8u) << 6) | ((v & 16u) << 8);
}

// key[e] = Morton index of the tile ray e = source * n_rays + i is in at substep k_mid (clamped to the grid, as its
// deposits are); hist[key]++
__global__ void ray_tile_key_kernel(uint32_t* key, uint32_t* hist, const float* sources, long long n, int n_rays, double ds,
                                 long long k_mid, int nx, int ny, int nz, int shift) {
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
        t[a] = uint32_t(int(c)) >> shift;
    }
    const uint32_t k = (spread5(t[0]) << 2) | (spread5(t[1]) << 1) | spread5(t[2]);
    key[e] = k;
    atomicAdd(hist + k, 1u);
}

// hist -> exclusive prefix sums (cursor), one block of 1024 threads, 32 consecutive keys per thread (all 32 loads in
// flight at once); hist itself is zeroed for the next call
__global__ void __launch_bounds__(1024) ray_tile_scan_kernel(uint32_t* hist, uint32_t* cursor) {
    constexpr int kPer = kRayTiles / 1024;
    __shared__ uint32_t warp_sum[32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint4* h4 = reinterpret_cast<uint4*>(hist + threadIdx.x * kPer);
    uint4 v[kPer / 4];
#pragma unroll
    for (int i = 0; i < kPer / 4; ++i) v[i] = h4[i];
    uint32_t sum = 0;
#pragma unroll
    for (int i = 0; i < kPer / 4; ++i) sum += v[i].x + v[i].y + v[i].z + v[i].w;
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
    uint4* c4 = reinterpret_cast<uint4*>(cursor + threadIdx.x * kPer);
#pragma unroll
    for (int i = 0; i < kPer / 4; ++i) {
        uint4 c;
        c.x = run; run += v[i].x;
        c.y = run; run += v[i].y;
        c.z = run; run += v[i].z;
        c.w = run; run += v[i].w;
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
