// rt_api.cu — the C ABI of librtmarch.so (include/rtmarch.h): argument checks on the host, then kernel
// launches on the caller's stream.  No torch types, no global state besides a thread-local error string.
#include "../../include/rtmarch.h"

#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>

#include "rt_ceiling_kernels.cuh"
#include "rt_march_kernels.cuh"

namespace {

thread_local char g_cuda_msg[256] = "no CUDA error recorded";

int cuda_fail(cudaError_t e, const char* where) {
    snprintf(g_cuda_msg, sizeof g_cuda_msg, "%s: %s", where, cudaGetErrorString(e));
    return RT_ECUDA;
}
#define RT_CUDA(call)                                       \
    do {                                                    \
        cudaError_t e_ = (call);                            \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call); \
    } while (0)

bool positive_finite(float v) { return std::isfinite(v) && v > 0.0f; }

// PAPER.md:25, D6.  Returns N_s, or -1 if it does not fit 31 bits.
long long substeps(float step_size, float c, float dt) {
    const double r = double(c) * double(dt) / double(step_size);
    if (!(r < 2147483647.0)) return -1;
    const double rr = std::nearbyint(r);
    if (rr >= 1.0 && std::fabs(r - rr) <= 1e-6 * r) return (long long)rr;
    return (long long)std::ceil(r);
}

// band of the coherent ray order: a power of two near sqrt(100 N_Omega), in [32, 1024]
int order_band(int n_rays) {
    const double target = std::sqrt(100.0 * double(n_rays));
    int lg = int(std::lround(std::log2(target)));
    lg = lg < 5 ? 5 : (lg > 10 ? 10 : lg);
    return 1 << lg;
}
int ray_slots(int n_rays) {
    const int band = order_band(n_rays);
    return int(((long long)n_rays + band - 1) / band) * band;
}

struct Checked {
    long long n_sub, cells;
};

int check_args(const void* j, const void* kappa, int nx, int ny, int nz, const void* sources, int n_src, int n_rays,
               int n_bins, float step_size, float c, float dt, int n_steps, const void* out, Checked* ck) {
    if (!j || !kappa || !sources || !out) return RT_EINVAL;
    if (nx < 1 || ny < 1 || nz < 1 || n_src < 1 || n_rays < 1 || n_bins < 1 || n_steps < 1) return RT_EINVAL;
    if (!positive_finite(step_size) || !positive_finite(c) || !positive_finite(dt)) return RT_EINVAL;
    if (n_rays > (1 << 30)) return RT_EINVAL;
    const long long cells = (long long)nx * ny;
    if (cells > 2147483647LL || cells * nz > 2147483647LL || cells * nz * n_bins > 2147483647LL) return RT_EINVAL;
    const long long ns = substeps(step_size, c, dt);
    if (ns < 1) return RT_EINVAL;
    const long long total = ns * n_steps;
    if (total > 2147483647LL) return RT_EINVAL;
    if (double(total) * double(step_size) > 268435456.0) return RT_EINVAL;   // path <= 2^28 cells
    if ((uintptr_t(j) | uintptr_t(kappa) | uintptr_t(out) | uintptr_t(sources)) & 3u) return RT_EALIGN;
    ck->n_sub = ns;
    ck->cells = cells * nz * n_bins;
    return RT_OK;
}

template <int NB>
int launch_march(const rt::MarchParams& P, int variant, cudaStream_t st) {
    const int threads = 128;
    const long long chunks = (P.n_slots + threads - 1) / threads;
    const long long blocks = chunks * P.n_groups * P.n_src;
    if (blocks > 2147483647LL) return RT_EINVAL;
    const bool sliding = (variant == RT_VARIANT_DEFAULT || variant == RT_VARIANT_SLIDING_LATTICE);
    if (sliding)
        rt::march_sliding_kernel<NB><<<unsigned(blocks), threads, 0, st>>>(P);
    else
        rt::march_direct_kernel<NB><<<unsigned(blocks), threads, 0, st>>>(P);
    RT_CUDA(cudaGetLastError());
    return RT_OK;
}

int build_ray_order(int n_rays, uint32_t* order, cudaStream_t st) {
    const int band = order_band(n_rays);
    const int bands = ray_slots(n_rays) / band;
    rt::ray_order_kernel<<<bands, band, band * sizeof(unsigned long long), st>>>(order, n_rays, band);
    RT_CUDA(cudaGetLastError());
    return RT_OK;
}

int march_impl(const float* j, const float* kappa, int nx, int ny, int nz, const float* sources, int n_src, int n_rays,
               int n_bins, float step_size, float c, float dt, int n_steps, float* out, void* workspace,
               size_t workspace_bytes, void* stream, int variant) {
    Checked ck;
    const int rc = check_args(j, kappa, nx, ny, nz, sources, n_src, n_rays, n_bins, step_size, c, dt, n_steps, out, &ck);
    if (rc != RT_OK) return rc;
    if (variant < RT_VARIANT_DEFAULT || variant > RT_VARIANT_SLIDING_LATTICE) return RT_EINVAL;
    const bool coherent = (variant == RT_VARIANT_DEFAULT || variant == RT_VARIANT_DIRECT_COHERENT);
    const size_t need = rt_workspace_bytes(nx, ny, nz, n_src, n_rays, n_bins, n_steps);
    if (coherent && (!workspace || workspace_bytes < need || (uintptr_t(workspace) & 15u))) return RT_EWORKSPACE;

    cudaStream_t st = static_cast<cudaStream_t>(stream);
    rt::MarchParams P;
    P.j = j; P.kappa = kappa; P.sources = sources; P.out = out;
    P.nx = nx; P.ny = ny; P.nz = nz; P.nb = n_bins;
    P.n_src = n_src; P.n_rays = n_rays;
    P.n_steps = n_steps; P.n_sub = int(ck.n_sub);
    P.ds = double(step_size); P.ds_f = step_size;
    P.emis = float(double(step_size) * 4.0 * 3.14159265358979323846 / double(n_rays));
    P.snap_stride = ck.cells;
    if (coherent) {
        P.ray_order = static_cast<const uint32_t*>(workspace);
        P.n_slots = ray_slots(n_rays);
        const int rc2 = build_ray_order(n_rays, static_cast<uint32_t*>(workspace), st);
        if (rc2 != RT_OK) return rc2;
    } else {
        P.ray_order = nullptr;
        P.n_slots = n_rays;
    }
    RT_CUDA(cudaMemsetAsync(out, 0, size_t(ck.cells) * size_t(n_steps) * sizeof(float), st));   // D14: overwrite

    // 4 bins per thread with 16-byte reductions when the layout allows it, else one bin per thread
    const bool vec4 = (n_bins % 4 == 0) && !((uintptr_t(j) | uintptr_t(kappa) | uintptr_t(out)) & 15u);
    int rc3;
    if (vec4) {
        P.n_groups = n_bins / 4;
        rc3 = launch_march<4>(P, variant, st);
    } else {
        P.n_groups = n_bins;
        rc3 = launch_march<1>(P, variant, st);
    }
    if (rc3 != RT_OK) return rc3;
    if (n_steps > 1) {
        const int threads = 256;
        long long blocks = (ck.cells + threads - 1) / threads;
        if (blocks > 148 * 16) blocks = 148 * 16;
        rt::snapshot_prefix_kernel<<<unsigned(blocks), threads, 0, st>>>(out, ck.cells, n_steps);
        RT_CUDA(cudaGetLastError());
    }
    return RT_OK;
}

}  // namespace

extern "C" {

int rt_march(const float* j, const float* kappa, int nx, int ny, int nz, const float* sources, int n_src, int n_rays,
             int n_bins, float step_size, float c, float dt, int n_steps, float* out, void* workspace,
             size_t workspace_bytes, void* stream) {
    return march_impl(j, kappa, nx, ny, nz, sources, n_src, n_rays, n_bins, step_size, c, dt, n_steps, out, workspace,
                      workspace_bytes, stream, RT_VARIANT_DEFAULT);
}

int rt_march_single(const float* j, const float* kappa, int nx, int ny, int nz, const float* source_pos, int n_rays,
                    int n_bins, float step_size, float c, float dt, int n_steps, float* out, void* workspace,
                    size_t workspace_bytes, void* stream) {
    return march_impl(j, kappa, nx, ny, nz, source_pos, 1, n_rays, n_bins, step_size, c, dt, n_steps, out, workspace,
                      workspace_bytes, stream, RT_VARIANT_DEFAULT);
}

int rt_march_ex(const float* j, const float* kappa, int nx, int ny, int nz, const float* sources, int n_src, int n_rays,
                int n_bins, float step_size, float c, float dt, int n_steps, float* out, void* workspace,
                size_t workspace_bytes, void* stream, int variant) {
    return march_impl(j, kappa, nx, ny, nz, sources, n_src, n_rays, n_bins, step_size, c, dt, n_steps, out, workspace,
                      workspace_bytes, stream, variant);
}

int rt_march_host(const float* j, const float* kappa, int nx, int ny, int nz, const float* sources, int n_src,
                  int n_rays, int n_bins, float step_size, float c, float dt, int n_steps, float* out) {
    Checked ck;
    const int rc = check_args(j, kappa, nx, ny, nz, sources, n_src, n_rays, n_bins, step_size, c, dt, n_steps, out, &ck);
    if (rc != RT_OK) return rc;
    const size_t grid_b = size_t(ck.cells) * sizeof(float), out_b = grid_b * size_t(n_steps);
    const size_t src_b = size_t(n_src) * 3 * sizeof(float);
    const size_t ws_b = rt_workspace_bytes(nx, ny, nz, n_src, n_rays, n_bins, n_steps);
    float *dj = nullptr, *dk = nullptr, *ds = nullptr, *dout = nullptr;
    void* dws = nullptr;
    cudaStream_t st = nullptr;
    int result = RT_OK;
    cudaError_t e = cudaSuccess;
    auto ok = [&](cudaError_t err, const char* where) {
        if (err != cudaSuccess && result == RT_OK) result = cuda_fail(err, where);
        return err == cudaSuccess;
    };
    if (ok(cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking), "cudaStreamCreate") &&
        ok(cudaMalloc(&dj, grid_b), "cudaMalloc j") && ok(cudaMalloc(&dk, grid_b), "cudaMalloc kappa") &&
        ok(cudaMalloc(&ds, src_b), "cudaMalloc sources") && ok(cudaMalloc(&dout, out_b), "cudaMalloc out") &&
        ok(cudaMalloc(&dws, ws_b), "cudaMalloc workspace") &&
        ok(cudaMemcpyAsync(dj, j, grid_b, cudaMemcpyHostToDevice, st), "H2D j") &&
        ok(cudaMemcpyAsync(dk, kappa, grid_b, cudaMemcpyHostToDevice, st), "H2D kappa") &&
        ok(cudaMemcpyAsync(ds, sources, src_b, cudaMemcpyHostToDevice, st), "H2D sources")) {
        result = march_impl(dj, dk, nx, ny, nz, ds, n_src, n_rays, n_bins, step_size, c, dt, n_steps, dout, dws, ws_b,
                            st, RT_VARIANT_DEFAULT);
        if (result == RT_OK) {
            ok(cudaMemcpyAsync(out, dout, out_b, cudaMemcpyDeviceToHost, st), "D2H out");
            ok(cudaStreamSynchronize(st), "cudaStreamSynchronize");
        }
    }
    (void)e;
    if (st) cudaStreamSynchronize(st);
    cudaFree(dj); cudaFree(dk); cudaFree(ds); cudaFree(dout); cudaFree(dws);
    if (st) cudaStreamDestroy(st);
    return result;
}

size_t rt_workspace_bytes(int nx, int ny, int nz, int n_src, int n_rays, int n_bins, int n_steps) {
    if (nx < 1 || ny < 1 || nz < 1 || n_src < 1 || n_rays < 1 || n_bins < 1 || n_steps < 1 || n_rays > (1 << 30))
        return 0;
    return size_t(ray_slots(n_rays)) * sizeof(uint32_t);
}

int rt_substeps_per_step(float step_size, float c, float dt) {
    if (!positive_finite(step_size) || !positive_finite(c) || !positive_finite(dt)) return RT_EINVAL;
    const long long ns = substeps(step_size, c, dt);
    return ns < 1 ? RT_EINVAL : int(ns);
}

int rt_launch_count(int n_bins, int n_steps) {
    if (n_bins < 1 || n_steps < 1) return RT_EINVAL;
    return 2 + (n_steps > 1 ? 1 : 0);   // ray order, march, (snapshot prefix)
}

int rt_directions(int n_rays, double* nhat, void* stream) {
    if (n_rays < 1 || n_rays > (1 << 30) || !nhat) return RT_EINVAL;
    rt::directions_kernel<<<(n_rays + 255) / 256, 256, 0, static_cast<cudaStream_t>(stream)>>>(nhat, n_rays);
    RT_CUDA(cudaGetLastError());
    return RT_OK;
}

int rt_trace_ray(const float* j, const float* kappa, int nx, int ny, int nz, int n_bins, const float* source_pos,
                 int ray_index, int n_rays, float step_size, int n_sub, double* pos, float* trace_I, float* trace_T,
                 void* stream) {
    if (!j || !kappa || !source_pos || !pos || !trace_I || !trace_T) return RT_EINVAL;
    if (nx < 1 || ny < 1 || nz < 1 || n_bins < 1 || n_rays < 1 || n_rays > (1 << 30) || ray_index < 0 ||
        ray_index >= n_rays || n_sub < 1 || !positive_finite(step_size))
        return RT_EINVAL;
    if ((long long)nx * ny * nz * n_bins > 2147483647LL) return RT_EINVAL;
    rt::MarchParams P{};
    P.j = j; P.kappa = kappa; P.sources = source_pos; P.out = nullptr; P.ray_order = nullptr;
    P.nx = nx; P.ny = ny; P.nz = nz; P.nb = n_bins;
    P.n_src = 1; P.n_rays = n_rays; P.n_slots = n_rays; P.n_groups = 1; P.n_steps = 1; P.n_sub = n_sub;
    P.ds = double(step_size); P.ds_f = step_size; P.emis = step_size; P.snap_stride = 0;
    rt::trace_ray_kernel<<<1, 32, 0, static_cast<cudaStream_t>(stream)>>>(P, uint32_t(ray_index), n_sub, pos, trace_I,
                                                                         trace_T);
    RT_CUDA(cudaGetLastError());
    return RT_OK;
}

int rt_ray_slots(int n_rays) {
    if (n_rays < 1 || n_rays > (1 << 30)) return RT_EINVAL;
    return ray_slots(n_rays);
}

int rt_ray_order(int n_rays, unsigned int* order, void* stream) {
    if (n_rays < 1 || n_rays > (1 << 30) || !order) return RT_EINVAL;
    return build_ray_order(n_rays, order, static_cast<cudaStream_t>(stream));
}

int rt_bench_red_ceiling(int mode, float* grid, int nx, int ny, int nz, int n_bins, long long n_red, unsigned int seed,
                         long long* n_issued, void* stream) {
    if (!grid || mode < 0 || mode > 5 || nx < 2 || ny < 2 || nz < 2 || n_bins < 1 || n_red < 1) return RT_EINVAL;
    const long long elems = (long long)nx * ny * nz * n_bins;
    if (elems > 2147483647LL || elems < 32) return RT_EINVAL;
    const bool vec = (n_bins % 4 == 0) && !(uintptr_t(grid) & 15u);
    if (mode == 1 && (elems % 4 || (uintptr_t(grid) & 15u))) return RT_EALIGN;
    const int threads = 256, blocks = 148 * 8;
    // reductions (red instructions x lanes) one thread issues per iteration
    const long long per_iter = (mode == 2 || mode == 5) ? 8LL * (vec ? n_bins / 4 : n_bins) : 8LL;
    const long long lanes = (long long)threads * blocks;
    long long iters = (n_red + lanes * per_iter - 1) / (lanes * per_iter);
    if (iters > 2147483647LL) return RT_EINVAL;
    rt::CeilingParams P{grid, nx, ny, nz, n_bins, int(iters), seed};
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    switch (mode) {
        case 0: rt::red_ceiling_kernel<0, 1><<<blocks, threads, 0, st>>>(P); break;
        case 1: rt::red_ceiling_kernel<1, 4><<<blocks, threads, 0, st>>>(P); break;
        case 2:
            if (vec) rt::red_ceiling_kernel<2, 4><<<blocks, threads, 0, st>>>(P);
            else rt::red_ceiling_kernel<2, 1><<<blocks, threads, 0, st>>>(P);
            break;
        case 3: rt::red_ceiling_kernel<3, 1><<<blocks, threads, 0, st>>>(P); break;
        case 4: rt::red_ceiling_kernel<4, 1><<<blocks, threads, 0, st>>>(P); break;
        default:
            if (vec) rt::red_ceiling_kernel<5, 4><<<blocks, threads, 0, st>>>(P);
            else rt::red_ceiling_kernel<5, 1><<<blocks, threads, 0, st>>>(P);
    }
    RT_CUDA(cudaGetLastError());
    if (n_issued) *n_issued = iters * lanes * per_iter;
    return RT_OK;
}

const char* rt_strerror(int code) {
    switch (code) {
        case RT_OK: return "ok";
        case RT_EINVAL: return "invalid argument (null pointer, non-positive size or step, or a documented limit exceeded)";
        case RT_EWORKSPACE: return "workspace missing, misaligned or smaller than rt_workspace_bytes()";
        case RT_ECUDA: return g_cuda_msg;
        case RT_EALIGN: return "pointer not sufficiently aligned";
        default: return "unknown rtmarch error code";
    }
}

const char* rt_version(void) { return "rtmarch 0.1 (sm_100a; sliding-stencil RED march)"; }

}  // extern "C"
