// rt_brick.cuh — the fp32 SCRATCH of march_phased_kernel (sm_100a): window bricks, vector reductions, concurrent drain.
//
// WHY.  ncu on C2 (profiles/r02b): the march is bound by the L1/LSU data pipe, and three quarters of its wavefronts
// are the deposits -- every lane of a red.global.add is its own 32-byte sector on its way to the L2, whatever it
// carries.  A stencil slide flushes a PLANE of 2 x 2 pending sums (the deposit has the trilinear
// footprint), so the payload of one reduction can be the whole plane: red.global.add.v4.f32 / .v2.f32 (there is no
// vector form for f64).  That needs (a) the 4 voxels of a plane contiguous and 16-byte aligned wherever the stencil
// sits, and (b) fp32 sums that stay accurate.
//
// (a) LAYOUT.  The scratch grid is indexed by WINDOW: S[x][Y0][Z0][4] holds, for the 2 x 2 (y, z) window that starts at
// (y0, z0) = (Y0 - 1, Z0 - 1), its four voxels (y0, z0), (y0, z0+1), (y0+1, z0), (y0+1, z0+1) as one 16-byte BRICK;
// Y0 in [0, ny], Z0 in [0, nz], so every window of the padded index range [-1, N] has its own aligned brick (a voxel
// lies in four windows: its sum is spread over four bricks, 4.1 x the memory of the grid).  Then
//     x-slide:  the trailing x-plane (2 x 2 in y, z)            -> 1 red.v4
//     y-slide:  per x slot, the z pair of the trailing y row    -> 2 red.v2  (the window that starts at that row)
//     z-slide:  per x slot, the y pair of the trailing z column -> 2 red.v4 {a, 0, b, 0}
// 1.67 reductions per slide instead of 4, and a brick's address is the lane's window offset, kept incrementally.
// Windows that start one z apart are neighbours in memory, so rays from z-adjacent sources (the lanes of a warp are
// sorted sources) share 32-byte sectors.  Index -1 and N (a clamped axis: both stencil indices are the same voxel,
// the other element of the pair carries an exact zero) are padding and only ever receive zeros.
//
// (b) ACCURACY.  A voxel's fp32 sum must not collect too many addends (stagnation at the hot voxels).
// Every block, when its rays are done, DRAINS one slice of the scratch into the fp64 accumulation grid:
// atom.exch.b32(element, 0) takes the element's sum and zeroes it in one indivisible step -- a reduction that arrives
// before the exchange is in the value taken, one that arrives after stays for the next drain, none is lost -- and
// the value is added to the fp64 grid with red.global.add.f64.  The slices rotate with the block index so that the
// whole scratch is drained kDrainRounds times per launch; a last pass after the march takes what is left.
// (Vector reductions are performed element by element, so every access to an element is a 4-byte atomic.)
#pragma once
#include "rt_common.cuh"

namespace rt {

#ifndef RT_DRAIN_ROUNDS
#define RT_DRAIN_ROUNDS 16
#endif
constexpr int kDrainRounds = RT_DRAIN_ROUNDS;          // the scratch is drained about this often per march launch
constexpr long long kDrainMaxUnits = 1 << 16;   // 16-byte units (bricks) one block drains at most

struct BrickGeom {
    int wy, wz;                   // windows per column / row: ny + 1, nz + 1
    int sx, sy;                   // floats per step of x, of Y0 (a step of Z0 is 4)
    long long step_stride;        // floats per time step: nx * wy * wz * 4
};

__host__ __device__ inline BrickGeom brick_geom(int nx, int ny, int nz) {
    BrickGeom g;
    g.wy = ny + 1;
    g.wz = nz + 1;
    g.sy = g.wz * 4;
    g.sx = g.wy * g.sy;
    g.step_stride = (long long)nx * g.sx;
    return g;
}

__device__ __forceinline__ void red_v4(float* p, float a, float b, float c, float d) {
    if ((__float_as_uint(a) | __float_as_uint(b) | __float_as_uint(c) | __float_as_uint(d)) != 0u)
        asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}
__device__ __forceinline__ void red_v2(float* p, float a, float b) {
    if ((__float_as_uint(a) | __float_as_uint(b)) != 0u)
        asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(p), "f"(a), "f"(b) : "memory");
}

// Drain bricks [b_begin, b_end) of the scratch (all time steps: brick b = ((m * nx + x) * wy + Y0) * wz + Z0) into the
// fp64 grid master[m][x][y][z]; thread `t` of `n_threads` takes every n_threads-th brick, kDrainBatch at a time: the
// peeks of a batch are in flight together, then its exchanges, then its reductions (a thread waits for three round
// trips per batch instead of five per brick).
// CONCURRENT: safe while other blocks reduce into the same elements (see above).  An element that reads zero at the
// peek is left alone (whatever arrives later stays for the next drain or for the snapshots).
constexpr int kDrainBatch = 4;

__device__ __forceinline__ uint32_t drain_take(float* e, float seen) {
    uint32_t bits = 0u;
    if (seen != 0.0f) asm volatile("atom.global.exch.b32 %0, [%1], %2;" : "=r"(bits) : "l"(e), "r"(0u) : "memory");
    return bits;
}
__device__ __forceinline__ void drain_give(double* m, uint32_t bits) {
    if (bits != 0u) asm volatile("red.global.add.f64 [%0], %1;" ::"l"(m), "d"(double(__uint_as_float(bits))) : "memory");
}

__device__ __forceinline__ void drain_bricks(float* scratch, double* master, const BrickGeom& G, int nx, int ny, int nz,
                                             long long b_begin, long long b_end, int t, int n_threads) {
    for (long long b0 = b_begin + t; b0 < b_end; b0 += (long long)kDrainBatch * n_threads) {
        float4 peek[kDrainBatch];
#pragma unroll
        for (int q = 0; q < kDrainBatch; ++q) {
            const long long b = b0 + (long long)q * n_threads;
            peek[q] = b < b_end ? __ldcg(reinterpret_cast<const float4*>(scratch + 4 * b)) : make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        }
        uint32_t bits[kDrainBatch][4];
#pragma unroll
        for (int q = 0; q < kDrainBatch; ++q) {
            float* e = scratch + 4 * (b0 + (long long)q * n_threads);
            bits[q][0] = drain_take(e, peek[q].x);
            bits[q][1] = drain_take(e + 1, peek[q].y);
            bits[q][2] = drain_take(e + 2, peek[q].z);
            bits[q][3] = drain_take(e + 3, peek[q].w);
        }
#pragma unroll
        for (int q = 0; q < kDrainBatch; ++q) {
            if ((bits[q][0] | bits[q][1] | bits[q][2] | bits[q][3]) == 0u) continue;
            const long long b = b0 + (long long)q * n_threads;
            const long long r = b / G.wz;
            const int Z0 = int(b - r * G.wz);
            const long long mx = r / G.wy;                      // m * nx + x
            const int Y0 = int(r - mx * G.wy);
            double* row = master + mx * ((long long)ny * nz);
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int y = Y0 - 1 + (i >> 1), z = Z0 - 1 + (i & 1);
                if (uint32_t(y) >= uint32_t(ny) || uint32_t(z) >= uint32_t(nz)) continue;      // padding: only zeros arrive
                drain_give(row + (long long)y * nz + z, bits[q][i]);
            }
        }
    }
}

// The same for a scratch in the plain grid layout (four bins per thread: a voxel's bins are one red.v4.f32): units of 4
// floats [u_begin, u_end), element e of the scratch belongs to element e of the fp64 grid.
__device__ __forceinline__ void drain_plain(float* scratch, double* master, long long u_begin, long long u_end, int t,
                                            int n_threads) {
    for (long long u0 = u_begin + t; u0 < u_end; u0 += (long long)kDrainBatch * n_threads) {
        float4 peek[kDrainBatch];
#pragma unroll
        for (int q = 0; q < kDrainBatch; ++q) {
            const long long u = u0 + (long long)q * n_threads;
            peek[q] = u < u_end ? __ldcg(reinterpret_cast<const float4*>(scratch + 4 * u)) : make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        }
        uint32_t bits[kDrainBatch][4];
#pragma unroll
        for (int q = 0; q < kDrainBatch; ++q) {
            float* e = scratch + 4 * (u0 + (long long)q * n_threads);
            bits[q][0] = drain_take(e, peek[q].x);
            bits[q][1] = drain_take(e + 1, peek[q].y);
            bits[q][2] = drain_take(e + 2, peek[q].z);
            bits[q][3] = drain_take(e + 3, peek[q].w);
        }
#pragma unroll
        for (int q = 0; q < kDrainBatch; ++q) {
            double* m = master + 4 * (u0 + (long long)q * n_threads);
#pragma unroll
            for (int i = 0; i < 4; ++i) drain_give(m + i, bits[q][i]);
        }
    }
}

// What the march left in the scratch, read back voxel by voxel when the snapshots are formed (no pass of its own, no
// atomics: the march is over).  Brick scratch: voxel (x, y, z) is element (a, b) of the four windows (Y0, Z0) =
// (y + 1 - a, z + 1 - b).  `sm` = scratch of time step m.
__device__ __forceinline__ double brick_residue(const float* sm, const BrickGeom& G, int x, int y, int z) {
    const float* w = sm + (long long)x * G.sx + (long long)y * G.sy + 4ll * z;      // window (Y0, Z0) = (y, z)
    return double(w[3]) + double(w[4 + 2]) + double(w[G.sy + 1]) + double(w[G.sy + 4]);
}

// out[m] <- sum over m' <= m of (acc[m'] + what is left in the scratch of step m'): the per-step increments become
// the cumulative snapshots (D7), summed in fp64 and rounded once.  BRICK: window-brick scratch (one bin),
// else the plain grid, which may be `out` itself (an element is read before this thread overwrites it).  Only the
// first acc_steps time steps have anything in the fp64 grid (all of them, but for PhasedPlan::no_drain of rt_api.cu).
template <bool BRICK>
__global__ void snapshot_finalize_scratch_kernel(const double* acc, const float* scratch, float* out, long long stride,
                                                 int n_steps, BrickGeom G, int ny, int nz, int acc_steps) {
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < stride;
         e += (long long)gridDim.x * blockDim.x) {
        int x = 0, y = 0, z = 0;
        if (BRICK) {
            const long long r = e / nz;
            z = int(e - r * nz);
            x = int(r / ny);
            y = int(r - (long long)x * ny);
        }
        double run = 0.0;
        for (int m0 = 0; m0 < n_steps; m0 += 4) {      // four time steps' loads in flight (scratch may be out: the compiler
            double inc[4];                             // cannot move a load above the previous step's store itself)
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int m = m0 + i;
                inc[i] = 0.0;
                if (m < n_steps) {
                    inc[i] = BRICK ? brick_residue(scratch + m * G.step_stride, G, x, y, z) : double(scratch[m * stride + e]);
                    if (m < acc_steps) inc[i] += acc[m * stride + e];
                }
            }
#pragma unroll
            for (int i = 0; i < 4; ++i)
                if (m0 + i < n_steps) {
                    run += inc[i];
                    out[(m0 + i) * stride + e] = float(run);
                }
        }
    }
}

// rt_march_step: out = (accumulate ? out : 0) + float(increment), increment = acc + what is left in the scratch
template <bool BRICK>
__global__ void step_finalize_scratch_kernel(const double* acc, const float* scratch, float* out, long long n, int accumulate,
                                             BrickGeom G, int ny, int nz) {
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x) {
        double inc = acc ? acc[e] : 0.0;
        if (BRICK) {
            const long long r = e / nz;
            const int z = int(e - r * nz), x = int(r / ny), y = int(r - (long long)x * ny);
            inc += brick_residue(scratch, G, x, y, z);
        } else {
            inc += double(scratch[e]);
        }
        out[e] = float((accumulate ? double(out[e]) : 0.0) + inc);
    }
}

}  // namespace rt
