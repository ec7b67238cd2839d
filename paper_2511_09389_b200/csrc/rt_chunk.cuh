// rt_chunk.cuh — the chunked march of grids far larger than the L2 (sm_100a): the rays of ALL sources advance
// together, a chunk of substeps per launch, and before every launch they are sorted by the tile of the grid they are
// in, so that the blocks in flight load and reduce into one neighbourhood of the grid instead of all of it.
//
// Eq. (2) fixes the order of the substeps of ONE ray only; rays are independent, so any
// interleaving of rays gives the same sums.  march_phased_kernel<.., STEP> already marches a ray from substep k0 with
// (I, exp(-tau)) carried in a state array (rt_march_step, D17); here the launches are chunks of a time
// step, the thread -> ray map is the sorted list (MarchParams::perm), and the state lives in the workspace.
// The sort is a locality heuristic: keys are computed in double, not in the march's fixed point, and the order of rays
// within a tile is whatever the scatter's atomics give -- neither changes a deposit.
#pragma once
#include "rt_common.cuh"

namespace rt {

struct ChunkGeom {
    int shift;               // a tile is (1 << shift)^3 cells
    int tx, ty, tz;          // tiles per axis (each <= 32)
    int n_tiles;             // Morton-coded: 32768 slots, most of them empty on small or flat grids
};

__host__ __device__ inline ChunkGeom chunk_geom(int nx, int ny, int nz) {
    ChunkGeom g;
    int m = nx > ny ? nx : ny;
    m = m > nz ? m : nz;
    g.shift = 3;
    while (((m - 1) >> g.shift) >= 32) ++g.shift;
    g.tx = ((nx - 1) >> g.shift) + 1;
    g.ty = ((ny - 1) >> g.shift) + 1;
    g.tz = ((nz - 1) >> g.shift) + 1;
    g.n_tiles = 32768;
    return g;
}

__device__ __forceinline__ uint32_t spread5(uint32_t v) {      // 5 bits -> every third bit
    return (v & 1u) | ((v & 2u) << 2) | ((v & 4u) << 4) | ((v & 8u) << 6) | ((v & 16u) << 8);
}

// key[e] = Morton index of the tile ray e = source * n_rays + i is in at substep k_mid (clamped to the grid, as its
// deposits are); hist[key]++
__global__ void chunk_key_kernel(uint32_t* key, uint32_t* hist, const float* sources, long long n, int n_rays, double ds,
                                 long long k_mid, int nx, int ny, int nz, ChunkGeom g) {
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
    const uint32_t k = (spread5(t[0]) << 2) | (spread5(t[1]) << 1) | spread5(t[2]);
    key[e] = k;
    atomicAdd(hist + k, 1u);
}

// hist -> exclusive prefix sums (cursor), one block; hist itself is zeroed for the next chunk
__global__ void chunk_scan_kernel(uint32_t* hist, uint32_t* cursor, int n_tiles) {
    __shared__ uint32_t part[1024];
    const int per = (n_tiles + blockDim.x - 1) / blockDim.x;
    const int b = threadIdx.x * per, e = min(b + per, n_tiles);
    uint32_t sum = 0;
    for (int t = b; t < e; ++t) sum += hist[t];
    part[threadIdx.x] = sum;
    __syncthreads();
    for (int d = 1; d < int(blockDim.x); d <<= 1) {
        const uint32_t v = (int(threadIdx.x) >= d) ? part[threadIdx.x - d] : 0u;
        __syncthreads();
        part[threadIdx.x] += v;
        __syncthreads();
    }
    uint32_t run = part[threadIdx.x] - sum;
    for (int t = b; t < e; ++t) {
        const uint32_t h = hist[t];
        cursor[t] = run;
        run += h;
        hist[t] = 0u;
    }
}

__global__ void chunk_scatter_kernel(uint32_t* perm, const uint32_t* key, uint32_t* cursor, long long n) {
    const long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (e >= n) return;
    perm[atomicAdd(cursor + key[e], 1u)] = uint32_t(e);
}

}  // namespace rt
