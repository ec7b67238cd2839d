// rt_ceiling_kernels.cuh — reduction-throughput microbenchmarks: the "measured L2-atomic roofline" the
// march kernel is set against (BASELINE.json metric).  Bench only; nothing here is on the
// march path.  Every thread keeps 8 independent reductions in flight per iteration.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace rt {

__device__ __forceinline__ uint32_t mix32(uint32_t x) {   // integer finaliser (avalanche)
    x ^= x >> 16; x *= 0x7feb352du;
    x ^= x >> 15; x *= 0x846ca68bu;
    x ^= x >> 16;
    return x;
}
__device__ __forceinline__ uint32_t xorshift32(uint32_t& s) {
    s ^= s << 13; s ^= s >> 17; s ^= s << 5;
    return s;
}
__device__ __forceinline__ uint32_t below(uint32_t r, uint32_t n) { return uint32_t((uint64_t(r) * n) >> 32); }

__device__ __forceinline__ void red1(float* p, float v) {
    asm volatile("red.global.add.f32 [%0], %1;" ::"l"(p), "f"(v) : "memory");
}
__device__ __forceinline__ void red4(float* p, float v) {
    asm volatile("red.global.add.v4.f32 [%0], {%1, %1, %1, %1};" ::"l"(p), "f"(v) : "memory");
}

__device__ __forceinline__ void red1d(double* p, double v) {
    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(p), "d"(v) : "memory");
}

struct CeilingParams {
    float* grid;                 // doubles for the fp64 modes
    int nx, ny, nz, nb;
    int iters;
    uint32_t seed;
};

// 8 corners of the stencil at base voxel (x,y,z): scalar reds (VEC == 1, bin 0..nb-1 each) or nb/4 v4 reds
template <int VEC>
__device__ __forceinline__ void red_stencil(const CeilingParams& P, int x, int y, int z, float v) {
    const size_t sy = size_t(P.nz) * P.nb, sx = sy * P.ny;
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        float* p = P.grid + (x + (c >> 2)) * sx + (y + ((c >> 1) & 1)) * sy + size_t(z + (c & 1)) * P.nb;
        if (VEC == 1) {
            for (int b = 0; b < P.nb; ++b) red1(p + b, v);
        } else {
            for (int b = 0; b < P.nb; b += 4) red4(p + b, v);
        }
    }
}

template <int MODE, int VEC>
__global__ void __launch_bounds__(256) red_ceiling_kernel(const CeilingParams P) {
    const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t s = mix32(tid * 2654435761u + P.seed) | 1u;
    const uint32_t n_elem = uint32_t(P.nx) * P.ny * P.nz * P.nb;
    const float v = 1.0f;
    if (MODE == 0) {            // M1: scalar, uniformly random
        for (int it = 0; it < P.iters; ++it)
#pragma unroll
            for (int u = 0; u < 8; ++u) red1(P.grid + below(xorshift32(s), n_elem), v);
    } else if (MODE == 1) {     // M2: v4, uniformly random, 16-byte aligned
        for (int it = 0; it < P.iters; ++it)
#pragma unroll
            for (int u = 0; u < 8; ++u) red4(P.grid + 4 * size_t(below(xorshift32(s), n_elem / 4)), v);
    } else if (MODE == 2) {     // M3: trilinear stencil at a random base voxel
        for (int it = 0; it < P.iters; ++it) {
            const int x = below(xorshift32(s), P.nx - 1), y = below(xorshift32(s), P.ny - 1),
                      z = below(xorshift32(s), P.nz - 1);
            red_stencil<VEC>(P, x, y, z, v);
        }
    } else if (MODE == 3) {     // M4: one address
        for (int it = 0; it < P.iters; ++it)
#pragma unroll
            for (int u = 0; u < 8; ++u) red1(P.grid, v);
    } else if (MODE == 4) {     // M5: warp-coalesced, random 128-byte line per warp instruction
        uint32_t ws = mix32((tid >> 5) * 2654435761u + P.seed) | 1u;
        for (int it = 0; it < P.iters; ++it)
#pragma unroll
            for (int u = 0; u < 8; ++u) red1(P.grid + 32 * size_t(below(xorshift32(ws), n_elem / 32)) + (tid & 31), v);
    } else if (MODE == 8) {     // M4b: every reduction to one of the 8 corner voxels of the grid (clamped far field)
        const size_t sy = size_t(P.nz) * P.nb, sx = sy * P.ny;
        for (int it = 0; it < P.iters; ++it)
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const uint32_t r = xorshift32(s);
                red1(P.grid + ((r & 1) ? (P.nx - 1) * sx : 0) + ((r & 2) ? (P.ny - 1) * sy : 0) +
                         ((r & 4) ? size_t(P.nz - 1) * P.nb : 0), v);
            }
    } else if (MODE == 9) {     // M4c: uniformly random voxels of the boundary shell (where clamped rays deposit)
        const size_t sy = size_t(P.nz) * P.nb, sx = sy * P.ny;
        for (int it = 0; it < P.iters; ++it)
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                int x = below(xorshift32(s), P.nx), y = below(xorshift32(s), P.ny), z = below(xorshift32(s), P.nz);
                const uint32_t f = below(xorshift32(s), 6);
                if (f == 0) x = 0; else if (f == 1) x = P.nx - 1; else if (f == 2) y = 0;
                else if (f == 3) y = P.ny - 1; else if (f == 4) z = 0; else z = P.nz - 1;
                red1(P.grid + x * sx + y * sy + size_t(z) * P.nb, v);
            }
    } else if (MODE == 6) {     // M1 in fp64: scalar, uniformly random
        double* g = reinterpret_cast<double*>(P.grid);
        for (int it = 0; it < P.iters; ++it)
#pragma unroll
            for (int u = 0; u < 8; ++u) red1d(g + below(xorshift32(s), n_elem), 1.0);
    } else if (MODE == 7) {     // M3 in fp64: trilinear stencil at a random base voxel, nb scalar reds per corner
        double* g = reinterpret_cast<double*>(P.grid);
        const size_t sy = size_t(P.nz) * P.nb, sx = sy * P.ny;
        for (int it = 0; it < P.iters; ++it) {
            const int x = below(xorshift32(s), P.nx - 1), y = below(xorshift32(s), P.ny - 1),
                      z = below(xorshift32(s), P.nz - 1);
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                double* p = g + (x + (c >> 2)) * sx + (y + ((c >> 1) & 1)) * sy + size_t(z + (c & 1)) * P.nb;
                for (int b = 0; b < P.nb; ++b) red1d(p + b, 1.0);
            }
        }
    } else {                    // M6: stencil along a random walk of half a cell per step
        float px = float(below(xorshift32(s), P.nx - 1)), py = float(below(xorshift32(s), P.ny - 1)),
              pz = float(below(xorshift32(s), P.nz - 1));
        float dx = float(int(xorshift32(s) >> 8) - (1 << 23)), dy = float(int(xorshift32(s) >> 8) - (1 << 23)),
              dz = float(int(xorshift32(s) >> 8) - (1 << 23));
        const float inv = 0.5f * rsqrtf(dx * dx + dy * dy + dz * dz + 1.0f);
        dx *= inv; dy *= inv; dz *= inv;
        for (int it = 0; it < P.iters; ++it) {
            int x = int(px), y = int(py), z = int(pz);
            if (px < 0.f || py < 0.f || pz < 0.f || x >= P.nx - 1 || y >= P.ny - 1 || z >= P.nz - 1) {
                px = float(below(xorshift32(s), P.nx - 1)); py = float(below(xorshift32(s), P.ny - 1));
                pz = float(below(xorshift32(s), P.nz - 1));
                x = int(px); y = int(py); z = int(pz);
            }
            red_stencil<VEC>(P, x, y, z, v);
            px += dx; py += dy; pz += dz;
        }
    }
}

}  // namespace rt
