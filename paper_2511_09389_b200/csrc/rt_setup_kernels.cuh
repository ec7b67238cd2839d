// rt_setup_kernels.cuh — the small kernels around the march: ray order, source order, direction dump (test
// hook), and the finalisation of the accumulation grid into cumulative fp32 snapshots.
#pragma once
#include "rt_common.cuh"

namespace rt {

// Coherent ray order.  Consecutive lattice indices share a latitude band but sit a golden angle apart in
// azimuth; sorting each band of M consecutive indices by azimuth makes every 32 consecutive slots (a warp)
// a compact patch of the sphere.  One block per band, bitonic sort of (azimuth fraction, index) keys.
__global__ void ray_order_kernel(uint32_t* order, int n_rays, int band) {
    extern __shared__ unsigned long long keys[];
    const uint32_t i = blockIdx.x * uint32_t(band) + threadIdx.x;
    const uint64_t turn = golden_turn64(i);
    keys[threadIdx.x] = (i < uint32_t(n_rays)) ? ((turn & 0xFFFFFFFF00000000ull) | i) : ~0ull;
    __syncthreads();
    for (int size = 2; size <= band; size <<= 1)
        for (int stride = size >> 1; stride > 0; stride >>= 1) {
            const int t = threadIdx.x, partner = t ^ stride;
            if (partner > t) {
                const unsigned long long a = keys[t], b = keys[partner];
                const bool up = (t & size) == 0;
                if ((a > b) == up) { keys[t] = b; keys[partner] = a; }
            }
            __syncthreads();
        }
    const unsigned long long kq = keys[threadIdx.x];
    order[i] = (kq == ~0ull) ? kPad : uint32_t(kq & 0xFFFFFFFFull);
}

// Spatial source order: rank of every source by the linear index of the (clamped) cell it sits in, ties by
// source index.  Consecutive ranks are then neighbours along z, then y, then x, so the 32 parallel rays of a
// map_src warp touch adjacent voxels (a Morton order was measured 9 % slower on C2: z-runs share sectors).
// O(n_src^2) comparisons (n_src <= 65536).
__device__ __forceinline__ unsigned long long source_cell_key(const float* sources, int s, int nx, int ny, int nz) {
    const float x = __ldg(sources + 3 * size_t(s)), y = __ldg(sources + 3 * size_t(s) + 1),
                z = __ldg(sources + 3 * size_t(s) + 2);
    const long long ix = (long long)fminf(fmaxf(floorf(x), 0.0f), float(nx - 1));
    const long long iy = (long long)fminf(fmaxf(floorf(y), 0.0f), float(ny - 1));
    const long long iz = (long long)fminf(fmaxf(floorf(z), 0.0f), float(nz - 1));
    return (unsigned long long)((ix * ny + iy) * nz + iz);
}

// one WARP per source: the lanes split the comparison loop, then add up their counts
__global__ void src_order_kernel(uint32_t* order, const float* sources, int n_src, int nx, int ny, int nz) {
    const int s = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (s >= n_src) return;
    const unsigned long long key = source_cell_key(sources, s, nx, ny, nz);
    uint32_t rank = 0;
    for (int t = lane; t < n_src; t += 32) {
        const unsigned long long kt = source_cell_key(sources, t, nx, ny, nz);
        rank += (kt < key) | ((kt == key) & (t < s));
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) rank += __shfl_xor_sync(0xFFFFFFFFu, rank, d);
    if (lane == 0) order[rank] = uint32_t(s);
}

__global__ void directions_kernel(double* nhat, int n_rays) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_rays) return;
    double nh[3];
    fib_direction(uint32_t(i), uint32_t(n_rays), nh);
    nhat[3 * size_t(i)] = nh[0];
    nhat[3 * size_t(i) + 1] = nh[1];
    nhat[3 * size_t(i) + 2] = nh[2];
}

// out[m] <- acc[0] + ... + acc[m]: per-step increments become the cumulative snapshots (D7).
// ACC = float with acc == out: in place; ACC = double: the fp64 accumulation grid is summed in fp64 and rounded once.
// `copies` grids, `copy_stride` elements apart, are added first (march_sliding_kernel<..., COPIES> spreads its
// reductions over them).
template <typename ACC>
__global__ void snapshot_finalize_kernel(const ACC* acc, float* out, long long stride, int n_steps, int copies = 1,
                                         long long copy_stride = 0) {
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < stride;
         e += (long long)gridDim.x * blockDim.x) {
        ACC run = ACC(0);
        for (int m = 0; m < n_steps; ++m) {
            for (int c = 0; c < copies; ++c) run += acc[c * copy_stride + m * stride + e];
            out[m * stride + e] = float(run);
        }
    }
}

// master += scratch (+ scratch2); scratch = scratch2 = 0 (the batched fp32 path of rt_api.cu: fp32 reductions of one
// batch of sources are folded into the fp64 grid before that scratch grid is used again, so no fp32 sum grows past
// one batch)
__global__ void drain_kernel(double* master, float* scratch, float* scratch2, long long n) {
    const long long n4 = n / 4;
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n4;
         e += (long long)gridDim.x * blockDim.x) {
        const float4 v = reinterpret_cast<float4*>(scratch)[e];
        const float4 u = scratch2 ? reinterpret_cast<float4*>(scratch2)[e] : make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        const bool nv = v.x != 0.0f || v.y != 0.0f || v.z != 0.0f || v.w != 0.0f;
        const bool nu = u.x != 0.0f || u.y != 0.0f || u.z != 0.0f || u.w != 0.0f;
        if (nv || nu) {
            double2* m = reinterpret_cast<double2*>(master) + 2 * e;
            double2 a = m[0], b = m[1];
            a.x += double(v.x) + double(u.x); a.y += double(v.y) + double(u.y);
            b.x += double(v.z) + double(u.z); b.y += double(v.w) + double(u.w);
            m[0] = a; m[1] = b;
            if (nv) reinterpret_cast<float4*>(scratch)[e] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
            if (nu) reinterpret_cast<float4*>(scratch2)[e] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        }
    }
}

// rt_march_step: out = (accumulate ? out : 0) + float(increment), increment summed in fp64
__global__ void step_finalize_kernel(const double* master, float* out, long long n, int accumulate) {
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x)
        out[e] = float((accumulate ? double(out[e]) : 0.0) + master[e]);
}

// fresh ray state: I = 0, exp(-tau) = 1 (D11)
__global__ void state_reset_kernel(float* state_I, float* state_T, long long n) {
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x) {
        state_I[e] = 0.0f;
        state_T[e] = 1.0f;
    }
}

}  // namespace rt

