// rt_api.cu — the C ABI of librtmarch.so (include/rtmarch.h): argument checks on the host, then kernel
// launches on the caller's stream.  No torch types; the only state kept between calls is a thread-local error
// string and rt_march_host's per-device memory pool.
#include "../../include/rtmarch.h"

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <shared_mutex>

#include "rt_ceiling_kernels.cuh"
#include "rt_march_direct.cuh"
#include "rt_adjoint.cuh"
#include "rt_brick.cuh"
#include "rt_ray_sort.cuh"
#include "rt_march_phased.cuh"
#include "rt_march_sliding.cuh"
#include "rt_setup_kernels.cuh"

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

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// workspace layout: [ray order: slots u32][source order: n_src u32][flag][fp64 accumulation grid x copies][fp32 scratch]
// [fp32 window-brick scratch of the one-bin phased march][sorted ray list of marches over grids beyond the L2]
struct Workspace {
    size_t src_order_at, flag_at, acc_at, scratch2_at, brick_at, brick_bytes, sort_at, sort_bytes, total;
    int acc_copies;
};
// One-bin calls deposit into an fp32 brick scratch (rt_brick.cuh): one 16-byte brick per 2 x 2 (y, z) window of each
// time step's grid, ~4.1 x the fp32 grid; the phased march is used while that stays below kBrickScratchLimit
constexpr size_t kBrickScratchLimit = size_t(1) << 30;
size_t brick_scratch_bytes(int nx, int ny, int nz, int n_steps, int n_bins) {
    if (n_bins != 1) return 0;
    const rt::BrickGeom g = rt::brick_geom(nx, ny, nz);
    const double bytes = double(g.step_stride) * double(n_steps) * sizeof(float);
    return bytes <= double(kBrickScratchLimit) ? size_t(g.step_stride) * size_t(n_steps) * sizeof(float) : 0;
}
bool use_batched_fp32(long long cells, int n_steps, int n_bins);
size_t ray_sort_bytes(int nx, int ny, int nz, int n_src, int n_rays, int n_steps, int n_bins);
size_t near_state_bytes(long long rays, int n_bins);
// One-bin-per-thread marches with fp64 reductions (the kernels of the non-default variants and of substeps of a cell or
// more) spread them over up to 4 copies of the grid, 48 MiB in all
constexpr size_t kAccCopiesBytes = size_t(48) << 20;
Workspace workspace_layout(int nx, int ny, int nz, int n_src, int n_rays, int n_steps, int n_bins) {
    Workspace w;
    const long long cells = (long long)nx * ny * nz * n_bins;
    const size_t grid = size_t(cells) * size_t(n_steps) * sizeof(double);
    w.acc_copies = use_batched_fp32(cells, n_steps, n_bins) ? 1 : int(std::min<size_t>(4, std::max<size_t>(1, kAccCopiesBytes / grid)));
    w.src_order_at = align_up(size_t(ray_slots(n_rays)) * sizeof(uint32_t), 16);
    w.flag_at = align_up(w.src_order_at + size_t(n_src) * sizeof(uint32_t), 16);      // same-fraction flag (weight-table march)
    w.acc_at = align_up(w.flag_at + 16, 256);
    w.scratch2_at = align_up(w.acc_at + grid * size_t(w.acc_copies), 256);
    // the batched fp32 path marches two batches at a time: `out` and this second fp32 grid are their scratch grids
    w.brick_at = align_up(w.scratch2_at + (use_batched_fp32(cells, n_steps, n_bins) ? size_t(cells) * size_t(n_steps) * sizeof(float) : 0), 256);
    w.brick_bytes = brick_scratch_bytes(nx, ny, nz, n_steps, n_bins);
    w.sort_at = align_up(w.brick_at + w.brick_bytes, 256);
    w.sort_bytes = ray_sort_bytes(nx, ny, nz, n_src, n_rays, n_steps, n_bins);
    w.total = w.sort_at + w.sort_bytes;
    return w;
}

// overlap_previous: programmatic stream serialization -- this grid may start while the tail of the previous kernel
// of the stream (a march_sliding_kernel<4, ...> it does not depend on) is still running
template <int NB, typename ACC>
int launch_march(const rt::MarchParams& P, bool sliding, cudaStream_t st, bool overlap_previous = false) {
    const long long blocks = rt::march_blocks(P.n_src, P.n_slots, P.n_groups, P.map_src);
    if (blocks > 2147483647LL) return RT_EINVAL;
    const unsigned g = unsigned(blocks);
    if (overlap_previous) {
        if (!sliding || NB != 4 || P.kappa_trilinear || P.state_I) return RT_EINVAL;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(g);
        cfg.blockDim = dim3(rt::kThreads);
        cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        RT_CUDA(cudaLaunchKernelEx(&cfg, rt::march_sliding_kernel<NB, ACC, 4, false, false, false>, P,
                                   static_cast<float*>(nullptr), 0LL));
        return RT_OK;
    }
    if (sliding) {
        // registers: 1 bin per thread runs 8 blocks/SM (64 registers); 4 bins 4 blocks/SM (128 registers, 8 bytes spilled)
        constexpr int kMinBlocks = (NB == 1) ? 8 : 4;
        if (P.kappa_trilinear) rt::march_sliding_kernel<NB, ACC, 1, false, true><<<g, rt::kThreads, 0, st>>>(P);
        else if (P.state_I) rt::march_sliding_kernel<NB, ACC, kMinBlocks, true><<<g, rt::kThreads, 0, st>>>(P);
        else if (P.acc_copies > 1)
            rt::march_sliding_kernel<NB, ACC, kMinBlocks, false, false, false, true><<<g, rt::kThreads, 0, st>>>(P);
        else rt::march_sliding_kernel<NB, ACC, kMinBlocks, false><<<g, rt::kThreads, 0, st>>>(P);
    } else {
        rt::march_direct_kernel<NB, ACC><<<g, rt::kThreads, 0, st>>>(P);
    }
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

constexpr int kMaxSortedSources = 65536;   // above this the O(n^2) source sort is skipped (identity order)

// The batched fp32 path (4-bin kernels): a batch is a range of sources x a range of direction slots holding at most
// 2^17 rays; the batches' fp32 sums are folded into the fp64 grid one by one.  It is used when the fp32 scratch
// grid is small enough for the drains to be cheap; larger grids take the 1-bin kernel with fp64 reductions.
constexpr long long kBatchRays = 1LL << 17;
constexpr size_t kBatchedScratchLimit = size_t(128) << 20;
struct Batching {
    int src_per_batch, slots_per_batch;
};
Batching plan_batches(int n_src, int n_slots, bool map_src) {
    Batching b;
    if (map_src) b.src_per_batch = int(32 * std::max(1LL, kBatchRays / (32LL * n_slots)));
    else b.src_per_batch = int(std::max(1LL, kBatchRays / (long long)n_slots));
    b.src_per_batch = std::min(b.src_per_batch, map_src ? (n_src + 31) / 32 * 32 : n_src);
    long long sl = std::max(128LL, kBatchRays / b.src_per_batch) / 128 * 128;      // whole blocks of slots
    b.slots_per_batch = int(std::min<long long>(sl, n_slots));
    return b;
}
bool use_batched_fp32(long long cells, int n_steps, int n_bins) {
    return n_bins % 4 == 0 && size_t(cells) * size_t(n_steps) * sizeof(float) <= kBatchedScratchLimit;
}

constexpr int kVariantKappaTrilinear = 64;   // internal: rt_march_trilinear_kappa

// what a variant code means (rtmarch.h RT_VARIANT_*)
struct Plan {
    bool sliding, coherent, map_src, acc64, one_bin, ktri;
};
bool make_plan(int variant, int n_src, Plan* pl) {
    const int kind = variant & 15;
    if (variant < 0 || (variant & ~127) || kind > RT_VARIANT_SLIDING_BY_SOURCE) return false;
    pl->ktri = (variant & kVariantKappaTrilinear) != 0;
    if (pl->ktri && (variant & ~kVariantKappaTrilinear)) return false;      // only with the default kernel path
    pl->acc64 = !(variant & RT_VARIANT_FLAG_ACC_F32);
    pl->one_bin = (variant & RT_VARIANT_FLAG_ONE_BIN) != 0;
    pl->sliding = !(kind == RT_VARIANT_DIRECT || kind == RT_VARIANT_DIRECT_COHERENT);
    pl->coherent = !(kind == RT_VARIANT_DIRECT || kind == RT_VARIANT_SLIDING_LATTICE);
    pl->map_src = (kind == RT_VARIANT_SLIDING_BY_SOURCE) || (kind == RT_VARIANT_DEFAULT && n_src >= 32);
    return true;
}

// march_phased_kernel (rt_march_phased.cuh) marches the calls of rt_march proper: the default variant with substeps
// shorter than a cell (a substep crosses at most one plane per axis).  Where its deposits go:
//   kPhasedOneBin    one bin, brick scratch affordable: fp32 window bricks in the workspace, one vector reduction per
//                    stencil plane, drained into the fp64 grid during the march
//   kPhasedFourBins  bins in groups of four and an fp32 grid of at most kBatchedScratchLimit (it then largely stays in
//                    the L2): `out` is the fp32 scratch, a voxel's four bins are one red.v4.f32, drained likewise
//   kPhasedDirect64  everything else (other bin counts; grids far larger than the L2, where a scratch and its drains
//                    would only add HBM traffic: measured on C4, 42 -> 32 ms with a scratch in four forms against 26 ms
//                    without): one bin per thread, bins in adjacent lanes, red.global.add.f64 straight into the fp64 grid
constexpr int kPhasedNone = 0, kPhasedOneBin = 1, kPhasedFourBins = 4, kPhasedDirect64 = 3;
int phased_kind(int variant, float step_size, long long cells, int n_steps, int n_bins, size_t brick_bytes, bool aligned16) {
    if ((variant != RT_VARIANT_DEFAULT && variant != kVariantKappaTrilinear) || !(step_size < 1.0f)) return kPhasedNone;
    if (n_bins == 1 && brick_bytes) return kPhasedOneBin;
    if (n_bins % 4 == 0 && aligned16 && use_batched_fp32(cells, n_steps, n_bins)) return kPhasedFourBins;
    return kPhasedDirect64;
}
// SORTED (the workspace has a ray list, ray_sort_bytes): the grid is far larger than the L2 and the threads take their
// rays from the list sorted by tile (rt_ray_sort.cuh).  Bins in groups of four then deposit as in kPhasedFourBins -- with
// the traffic kept local the fp32 scratch pays again (C4: 17.3 ms, against 20.5 ms with red.global.add.f64 per bin and
// 25.4 ms with that and the rays by direction).
// NO_DRAIN: a sorted four-bin march whose elements collect few deposits -- on average at most kNoDrainDeposits per
// element and time step (a ray-substep deposits into 8 voxels; C4: 32) -- is not drained: on such a grid every drain
// round streams the scratch and read-modify-writes the fp64 grid through HBM (C4: 17 of the march's 33 GB).  What fp32
// sums cannot take are the voxels next to a SOURCE: all N_Omega rays of the source deposit there, with nearly the same
// addend each, and the rounding errors of equal addends do not cancel (measured on C4: up to 3.9e-4 relative at the 8
// voxels around each source with everything in fp32, everywhere else < 1e-5).  So the first near_substeps substeps of
// every ray -- while it is within R = 2 + sqrt(N_Omega / (1024 pi)) cells of its source, beyond which fewer than 256
// rays of the source meet in a voxel -- are a launch of their own that reduces into the fp64 grid (one bin per lane,
// red.global.add.f64), (I, exp(-tau)) go through a ray state in the workspace as in rt_march_step, and the four-bin
// launch marches the rest into the fp32 scratch.  Only the time steps those first substeps fall into have anything in
// the fp64 grid: only they are zeroed, and read when the snapshots are formed.
// And no element may collect too many addends: a ray sums its deposits into a voxel in registers while the voxel is in
// its stencil, so an element receives at most one addend per ray and time step -- also the corner and face voxels that
// rays outside the box keep depositing into -- i.e. at most n_src N_Omega of them.  The bound is that of
// two drain rounds (drain_rounds: one per 2^19 rays; on C2, sums of 2^21 rays' addends were off by 2e-4 at worst).
constexpr double kNoDrainDeposits = 256.0;
constexpr long long kNoDrainRays = 1LL << 21;
long long near_substeps(int n_rays, float step_size) {
    const double r = 2.0 + std::sqrt(double(n_rays) / (1024.0 * 3.14159265358979323846));
    return (long long)std::ceil(r / double(step_size));
}
struct PhasedPlan {
    int kind;
    bool sorted, no_drain;
};
PhasedPlan phased_plan(int variant, float step_size, long long cells, int n_steps, int n_bins, const Workspace& wl, bool aligned16,
                       bool one_bin_per_thread, double ray_substeps_per_step, long long near_k, long long n_sub) {
    PhasedPlan pp;
    pp.kind = phased_kind(variant, step_size, cells, n_steps, n_bins, wl.brick_bytes, aligned16);
    pp.sorted = pp.kind == kPhasedDirect64 && wl.sort_bytes != 0;
    if (pp.sorted && n_bins % 4 == 0 && aligned16) pp.kind = kPhasedFourBins;
    // the trilinear-kappa and the tangent march exist with one bin per thread only
    if (one_bin_per_thread && pp.kind == kPhasedFourBins) pp.kind = kPhasedDirect64;
    pp.no_drain = pp.sorted && pp.kind == kPhasedFourBins && near_k <= n_sub &&
                  ray_substeps_per_step * 8.0 <= kNoDrainDeposits * double(cells / n_bins) &&
                  ray_substeps_per_step <= double(kNoDrainRays) * double(n_sub);
    return pp;
}
// how often the scratch is drained during a march: an fp32 sum should not collect much more than 2^19 rays' deposits
// (C2, 8.6 M rays: 16 rounds, relative L2 error 6e-6 against 2.5e-5 with 4 rounds and 1.2e-4 with none)
int drain_rounds(long long n_rays_total) {
    return int(std::min<long long>(std::max<long long>(n_rays_total >> 19, 1), rt::kDrainRounds));
}

// the plan of RT_VARIANT_DEFAULT (make_plan cannot fail for it)
Plan default_plan(int n_src) {
    Plan pl{};
    const bool ok = make_plan(RT_VARIANT_DEFAULT, n_src, &pl);
    (void)ok;
    return pl;
}

// The launch parameters every march / adjoint entry shares: medium, geometry, substep constants (emission quadrature
// weight ds * 4 pi / N_Omega of D8, attenuation scale -ds log2 e), one launch covering all sources and direction slots.
rt::MarchParams base_params(const float* j, const float* kappa, int nx, int ny, int nz, const float* sources, int n_src,
                            int n_rays, int n_bins, float step_size, int n_steps, const Checked& ck, const Plan& pl) {
    rt::MarchParams P{};
    P.acc_copies = 1;
    P.j = j; P.kappa = kappa; P.sources = sources;
    P.nx = nx; P.ny = ny; P.nz = nz; P.nb = n_bins;
    P.n_src = n_src; P.src_begin = 0; P.slot_begin = 0; P.n_rays = n_rays;
    P.n_groups = n_bins;
    P.n_steps = n_steps; P.n_sub = int(ck.n_sub);
    P.ds = double(step_size); P.ds_f = step_size;
    P.emis = float(double(step_size) * 4.0 * 3.14159265358979323846 / double(n_rays));
    P.att_scale = float(-double(step_size) * 1.4426950408889634074);
    P.snap_stride = ck.cells;
    P.map_src = pl.map_src ? 1 : 0;
    P.kappa_trilinear = pl.ktri ? 1 : 0;
    P.n_slots = n_rays;
    return P;
}

// the coherent ray order and the spatial source order of a plan, built on the stream into the head of the workspace
int build_orders(rt::MarchParams& P, const Plan& pl, const Workspace& wl, char* ws, cudaStream_t st) {
    if (pl.coherent) {
        P.ray_order = reinterpret_cast<const uint32_t*>(ws);
        P.n_slots = ray_slots(P.n_rays);
        const int rc = build_ray_order(P.n_rays, reinterpret_cast<uint32_t*>(ws), st);
        if (rc != RT_OK) return rc;
    }
    if (pl.map_src && P.n_src <= kMaxSortedSources) {
        uint32_t* so = reinterpret_cast<uint32_t*>(ws + wl.src_order_at);
        rt::src_order_kernel<<<(P.n_src + 3) / 4, 128, 0, st>>>(so, P.sources, P.n_src, P.nx, P.ny, P.nz);
        RT_CUDA(cudaGetLastError());
        P.src_order = so;
    }
    return RT_OK;
}

// rt_march_step: one time step from substep k0 with the ray state carried in `state`
struct StepArgs {
    float* state;
    long long k0;
    int accumulate;
};

// rt_march_step with four bins per thread (phased_plan): the fp32 scratch grid behind the workspace
size_t step_scratch_bytes(long long cells, int n_bins) {
    return n_bins % 4 == 0 ? size_t(cells) * sizeof(float) : 0;
}

// Marches over grids far larger than the L2 -- the fp32 grid of all time steps beyond kBatchedScratchLimit, no brick
// scratch -- map their threads to rays through a list sorted by tile (rt_ray_sort.cuh).
// Workspace behind the brick scratch: [hist: kRayTiles u32][cursor: kRayTiles u32][ray state: 2 x rays x bins f32, bins in
// fours only][perm: rays u32][key: rays u32]
size_t ray_sort_bytes(int nx, int ny, int nz, int n_src, int n_rays, int n_steps, int n_bins) {
    const long long cells = (long long)nx * ny * nz * n_bins;
    if ((n_bins == 1 && brick_scratch_bytes(nx, ny, nz, n_steps, n_bins)) ||
        size_t(cells) * size_t(n_steps) * sizeof(float) <= kBatchedScratchLimit)
        return 0;
    const long long rays = (long long)n_src * n_rays;
    if (rays >= (1LL << 32)) return 0;
    return 2 * size_t(rt::kRayTiles) * sizeof(uint32_t) + near_state_bytes(rays, n_bins) + size_t(rays) * 2 * sizeof(uint32_t);
}
// (I, exp(-tau)) of every ray and bin between the two launches of a march that is not drained (phased_plan)
size_t near_state_bytes(long long rays, int n_bins) {
    return n_bins % 4 == 0 ? 2 * size_t(rays) * size_t(n_bins) * sizeof(float) : 0;
}

// the instantiation of march_phased_kernel for a deposit mode (phased_kind)
template <bool TABLE, bool STEP>
int launch_phased(const rt::MarchParams& P, int kind, unsigned blocks, cudaStream_t st) {
    // the plain one-bin march with 32 sources x ONE direction per warp (map_src = 1) has an instantiation of its own
    const bool one_dir = !TABLE && kind == kPhasedOneBin && P.map_src == 1;
    if (P.kappa_trilinear) {           // rt_march_trilinear_kappa: one bin per thread in both deposit modes
        if (STEP || P.dkappa || kind == kPhasedFourBins) return RT_EINVAL;
        if (one_dir) rt::march_phased_kernel<1, false, true, float, false, false, true, false, true><<<blocks, rt::kThreads, 0, st>>>(P);
        else if (kind == kPhasedOneBin) rt::march_phased_kernel<1, TABLE, true, float, false, false, true><<<blocks, rt::kThreads, 0, st>>>(P);
        else rt::march_phased_kernel<1, TABLE, false, double, false, false, true><<<blocks, rt::kThreads, 0, st>>>(P);
        RT_CUDA(cudaGetLastError());
        return RT_OK;
    }
    if (P.dkappa) {                    // rt_march_jvp_kappa: one bin per thread in both deposit modes
        if (STEP || kind == kPhasedFourBins) return RT_EINVAL;
        if (one_dir) rt::march_phased_kernel<1, false, true, float, false, true, false, false, true><<<blocks, rt::kThreads, 0, st>>>(P);
        else if (kind == kPhasedOneBin) rt::march_phased_kernel<1, TABLE, true, float, false, true><<<blocks, rt::kThreads, 0, st>>>(P);
        else rt::march_phased_kernel<1, TABLE, false, double, false, true><<<blocks, rt::kThreads, 0, st>>>(P);
        RT_CUDA(cudaGetLastError());
        return RT_OK;
    }
    if (one_dir) rt::march_phased_kernel<1, false, true, float, STEP, false, false, false, true><<<blocks, rt::kThreads, 0, st>>>(P);
    else if (kind == kPhasedOneBin) rt::march_phased_kernel<1, TABLE, true, float, STEP><<<blocks, rt::kThreads, 0, st>>>(P);
    else if (kind == kPhasedFourBins) rt::march_phased_kernel<4, TABLE, false, float, STEP><<<blocks, rt::kThreads, 0, st>>>(P);
    else rt::march_phased_kernel<1, TABLE, false, double, STEP><<<blocks, rt::kThreads, 0, st>>>(P);
    RT_CUDA(cudaGetLastError());
    return RT_OK;
}

// The two launches of a sorted four-bin march that is not drained (phased_plan): substeps [k0, k_near) one bin per lane
// into the fp64 grid, [k_near, k_end) four bins per thread into the fp32 scratch, (I, exp(-tau)) carried through a ray
// state -- the caller's (rt_march_step) or one in the workspace.  P: the parameters of the whole call, the ray list set.
int run_near_and_far(rt::MarchParams P, long long k_near, long long k_end, bool callers_state, char* state_ws, long long n_ray,
                     int n_bins, cudaStream_t st) {
    const int n_sub = P.n_sub;
    const long long k0 = P.k0;
    if (!callers_state) {
        P.state_I = reinterpret_cast<float*>(state_ws);
        P.state_T = P.state_I + n_ray * n_bins;
        rt::state_reset_kernel<<<148 * 8, 256, 0, st>>>(P.state_I, P.state_T, n_ray * n_bins);
    }
    P.drain_units_per_block = 0;
    if (k_near > k0) {                 // at most the first time steps of the call
        rt::MarchParams N = P;
        N.n_groups = n_bins;
        N.n_steps = int((k_near - k0 + n_sub - 1) / n_sub);
        N.first_left = 0;
        if (k_near < k_end) {          // ends inside a time step: march it as (whole steps, then) a short last step
            if (N.n_steps > 1) return RT_EINVAL;       // (near_substeps <= N_s is a condition of the plan)
            N.n_sub = int(k_near - k0);
        }
        const long long nb_ = rt::perm_blocks(n_ray, N.n_groups);
        if (nb_ > 2147483647LL) return RT_EINVAL;
        const int rc = launch_phased<false, true>(N, kPhasedDirect64, unsigned(nb_), st);
        if (rc != RT_OK) return rc;
    }
    if (k_near < k_end) {
        rt::MarchParams F = P;
        const long long into = (k_near - k0) % n_sub;            // substeps of its first time step already marched
        F.k0 = k_near;
        F.first_left = into ? int(n_sub - into) : 0;
        const long long skipped = (k_near - k0) / n_sub;         // whole time steps marched by the first launch
        F.n_steps = P.n_steps - int(skipped);
        F.acc = static_cast<double*>(P.acc) + skipped * P.snap_stride;
        F.scratch = P.scratch + skipped * P.snap_stride;
        const long long fb_ = rt::perm_blocks(n_ray, F.n_groups);
        if (fb_ > 2147483647LL) return RT_EINVAL;
        const int rc = launch_phased<false, true>(F, kPhasedFourBins, unsigned(fb_), st);
        if (rc != RT_OK) return rc;
    }
    return RT_OK;
}

// rt_march proper (and rt_march_step, rt_march_trilinear_kappa, rt_march_jvp_kappa) through march_phased_kernel: memsets,
// the thread -> ray map (ray and source order; or the sorted ray list), (fraction test, weight-table instantiation,)
// plain instantiation, snapshots.
int run_phased(rt::MarchParams P, const PhasedPlan& pp, const Plan& pl, const Workspace& wl, char* ws, double* master, float* out,
               size_t n_acc, long long cells, const StepArgs* step, int nx, int ny, int nz, const float* sources, int n_src,
               int n_rays, int n_bins, float step_size, int n_steps, cudaStream_t st) {
    const int fin_threads = 256;
    long long fin_blocks = (cells + fin_threads - 1) / fin_threads;
    if (fin_blocks > 148 * 16) fin_blocks = 148 * 16;
    const int phased = pp.kind;
    // The phased march deposits into an fp32 scratch -- window bricks in the workspace (one bin), or the plain grid
    // (four bins per thread; `out` itself, or for rt_march_step, whose `out` may hold the running field, a grid behind
    // the workspace) -- and drains it into the fp64 grid as it goes; or it reduces straight into the fp64 grid.  The
    // snapshots (the step's increment) are formed from the fp64 grid plus what the march left in the scratch.
    P.n_groups = phased == kPhasedFourBins ? n_bins / 4 : n_bins;
    P.acc = master;
    P.scratch = phased == kPhasedOneBin ? reinterpret_cast<float*>(ws + wl.brick_at)
                                        : (step ? reinterpret_cast<float*>(ws + wl.total) : out);
    const size_t scratch_bytes = phased == kPhasedDirect64 ? 0 : (phased == kPhasedOneBin ? wl.brick_bytes : n_acc * sizeof(float));
    P.n_drain_units = std::max<long long>(1, (long long)(scratch_bytes / 16));
    // not drained (phased_plan): the substeps [k0, k_near) of this call go into the fp64 grid in a launch of their own
    const long long k_end = P.k0 + (long long)P.n_sub * n_steps;
    const long long k_near = pp.no_drain ? std::min(std::max(near_substeps(n_rays, step_size), P.k0), k_end) : P.k0;
    const int acc_steps = pp.no_drain ? int((k_near - P.k0 + P.n_sub - 1) / P.n_sub) : n_steps;      // time steps with fp64 content
    if (acc_steps) RT_CUDA(cudaMemsetAsync(master, 0, size_t(cells) * size_t(acc_steps) * sizeof(double), st));
    if (scratch_bytes) RT_CUDA(cudaMemsetAsync(P.scratch, 0, scratch_bytes, st));
    const long long n_ray = (long long)n_src * n_rays;
    long long mb;
    if (pp.sorted) {
        // key = tile at the middle of the marched substeps, histogram, prefix sums, scatter
        uint32_t* hist = reinterpret_cast<uint32_t*>(ws + wl.sort_at);
        uint32_t* cursor = hist + rt::kRayTiles;
        uint32_t* perm = reinterpret_cast<uint32_t*>(reinterpret_cast<char*>(cursor + rt::kRayTiles) + near_state_bytes(n_ray, n_bins));
        uint32_t* key = perm + n_ray;
        const rt::RaySortGeom sg = rt::ray_sort_geom(nx, ny, nz);
        RT_CUDA(cudaMemsetAsync(hist, 0, size_t(sg.n_keys) * sizeof(uint32_t), st));
        const unsigned rb = unsigned((n_ray + 255) / 256);
        const long long k_mid = P.k0 + (long long)P.n_sub * n_steps / 2;
        rt::ray_tile_key_kernel<<<rb, 256, 0, st>>>(key, hist, sources, n_ray, n_rays, P.ds, k_mid, nx, ny, nz, sg);
        rt::ray_tile_scan_kernel<<<1, 1024, 0, st>>>(hist, cursor, sg.n_keys);
        rt::ray_tile_scatter_kernel<<<rb, 256, 0, st>>>(perm, key, cursor, n_ray);
        RT_CUDA(cudaGetLastError());
        P.map_src = 2;
        P.perm = perm;
        P.n_perm = n_ray;
        mb = rt::perm_blocks(n_ray, P.n_groups);
    } else {
        const int rco = build_orders(P, pl, wl, ws, st);
        if (rco != RT_OK) return rco;
        mb = rt::march_blocks(P.n_src, P.n_slots, P.n_groups, P.map_src);
    }
    if (mb > 2147483647LL) return RT_EINVAL;
    const long long per = (P.n_drain_units * drain_rounds(n_ray) + mb - 1) / mb;
    P.drain_units_per_block = std::min<long long>(std::max<long long>(per, 1), rt::kDrainMaxUnits);
    if (pp.no_drain) {
        const int rcn = run_near_and_far(P, k_near, k_end, step != nullptr, ws + wl.sort_at + 2 * rt::kRayTiles * sizeof(uint32_t), n_ray,
                                         n_bins, st);
        if (rcn != RT_OK) return rcn;
    } else {
        if (pl.map_src && !pp.sorted) {
            // Sources that share their cell fractions (decided on the device) take the weight-table instantiation, others
            // the plain one: both are launched, each returns at once when the flag says the call is the other's
            int* flag = reinterpret_cast<int*>(ws + wl.flag_at);
            rt::same_fraction_kernel<<<1, 256, 0, st>>>(flag, sources, n_src, step_size);
            P.same_frac = flag;
            const int rct = step ? launch_phased<true, true>(P, phased, unsigned(mb), st) : launch_phased<true, false>(P, phased, unsigned(mb), st);
            if (rct != RT_OK) return rct;
        }
        if (phased == kPhasedDirect64 && pl.map_src && !pp.sorted) {
            // sources in general position, fp64 reductions: warp = 32 (direction, bin) pairs of ONE source, so that the
            // blocks in flight stay around a few sources (the brick path is faster by sorted sources)
            P.map_src = 0;
            P.src_order = nullptr;
            mb = rt::march_blocks(P.n_src, P.n_slots, P.n_groups, 0);
            if (mb > 2147483647LL) return RT_EINVAL;
        }
        const int rcp = step ? launch_phased<false, true>(P, phased, unsigned(mb), st) : launch_phased<false, false>(P, phased, unsigned(mb), st);
        if (rcp != RT_OK) return rcp;
    }
    // the snapshots (the step's increment): the fp64 grid plus what the march left in the scratch, rounded once
    const rt::BrickGeom G = rt::brick_geom(nx, ny, nz);
    const unsigned fb = unsigned(fin_blocks);
    if (step) {
        if (phased == kPhasedOneBin)
            rt::step_finalize_scratch_kernel<true><<<fb, fin_threads, 0, st>>>(master, P.scratch, out, cells, step->accumulate, G, ny, nz);
        else if (phased == kPhasedFourBins)
            rt::step_finalize_scratch_kernel<false><<<fb, fin_threads, 0, st>>>(acc_steps ? master : nullptr, P.scratch, out, cells,
                                                                               step->accumulate, G, ny, nz);
        else
            rt::step_finalize_kernel<<<fb, fin_threads, 0, st>>>(master, out, cells, step->accumulate);
    } else {
        if (phased == kPhasedOneBin)
            rt::snapshot_finalize_scratch_kernel<true><<<fb, fin_threads, 0, st>>>(master, P.scratch, out, cells, n_steps, G, ny, nz, acc_steps);
        else if (phased == kPhasedFourBins)
            rt::snapshot_finalize_scratch_kernel<false><<<fb, fin_threads, 0, st>>>(master, P.scratch, out, cells, n_steps, G, ny, nz, acc_steps);
        else
            rt::snapshot_finalize_kernel<double><<<fb, fin_threads, 0, st>>>(master, out, cells, n_steps);
    }
    RT_CUDA(cudaGetLastError());
    return RT_OK;
}

int march_impl(const float* j, const float* kappa, int nx, int ny, int nz, const float* sources, int n_src, int n_rays,
               int n_bins, float step_size, float c, float dt, int n_steps, float* out, void* workspace,
               size_t workspace_bytes, void* stream, int variant, const StepArgs* step = nullptr,
               const float* dkappa = nullptr) {
    Checked ck;
    const int rc = check_args(j, kappa, nx, ny, nz, sources, n_src, n_rays, n_bins, step_size, c, dt, n_steps, out, &ck);
    if (rc != RT_OK) return rc;
    Plan pl;
    if (!make_plan(variant, n_src, &pl)) return RT_EINVAL;
    const Workspace wl = workspace_layout(nx, ny, nz, n_src, n_rays, n_steps, n_bins);
    const size_t need = wl.total + (step ? step_scratch_bytes(ck.cells, n_bins) : 0);
    if (!workspace || workspace_bytes < need || (uintptr_t(workspace) & 15u)) return RT_EWORKSPACE;
    char* ws = static_cast<char*>(workspace);
    if (step) {
        if (!step->state || (uintptr_t(step->state) & 15u)) return RT_EINVAL;
        const double last = double(step->k0) + double(ck.n_sub);
        if (step->k0 < 0 || last > 2147483647.0 || last * double(step_size) > 268435456.0) return RT_EINVAL;
    }

    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (pl.ktri && step) return RT_EINVAL;
    rt::MarchParams P = base_params(j, kappa, nx, ny, nz, sources, n_src, n_rays, n_bins, step_size, n_steps, ck, pl);
    P.state_I = step ? step->state : nullptr;
    P.state_T = step ? step->state + size_t(n_src) * size_t(n_rays) * size_t(n_bins) : nullptr;
    P.k0 = step ? step->k0 : 0;
    const size_t n_acc = size_t(ck.cells) * size_t(n_steps);
    double* master = reinterpret_cast<double*>(ws + wl.acc_at);
    const int fin_threads = 256;
    long long fin_blocks = (ck.cells + fin_threads - 1) / fin_threads;
    if (fin_blocks > 148 * 16) fin_blocks = 148 * 16;

    const bool aligned4 = (n_bins % 4 == 0) && !((uintptr_t(j) | uintptr_t(kappa) | uintptr_t(out)) & 15u);
    const PhasedPlan pp = phased_plan(variant, step_size, ck.cells, n_steps, n_bins, wl, aligned4, dkappa || pl.ktri,
                                      double(n_src) * double(n_rays) * double(ck.n_sub), near_substeps(n_rays, step_size), ck.n_sub);
    if (dkappa) {                      // the tangent march exists in the phased kernel only
        if (pp.kind == kPhasedNone || step || pl.ktri) return RT_EINVAL;
        P.dkappa = dkappa;
    }
    if (pp.kind != kPhasedNone)
        return run_phased(P, pp, pl, wl, ws, master, out, n_acc, ck.cells, step, nx, ny, nz, sources, n_src, n_rays, n_bins,
                          step_size, n_steps, st);
    const int rco = build_orders(P, pl, wl, ws, st);
    if (rco != RT_OK) return rco;
    // What is left: steps of a cell or more and the non-default variants, through march_sliding_kernel / march_kernel.
    // 4 bins per thread (16-byte loads, 16-byte fp32 reductions) when the layout allows it -- and, with fp64
    // accumulation, only on the batched path: there is no 16-byte fp64 reduction, and four scalar ones per voxel
    // make the 4-bin kernel reduction bound, so larger grids march one bin per thread (bins in adjacent lanes
    // share the sectors of their fp64 reductions)
    const bool batched = aligned4 && !pl.one_bin && pl.acc64 && pl.sliding && use_batched_fp32(ck.cells, n_steps, n_bins);
    const bool vec4 = aligned4 && !pl.one_bin && (batched || !pl.acc64 || !pl.sliding);
    P.n_groups = vec4 ? n_bins / 4 : n_bins;

    if (batched) {
        // `out` (rt_march_step: a grid behind the fp64 grid, it may be accumulating into out) is the fp32 scratch
        // grid of ONE batch: no fp32 sum ever holds more than 2^17 rays, which bounds the error of fp32
        // accumulation; after every batch drain_kernel folds it into the fp64 grid and zeroes it.
        float* scratch = step ? reinterpret_cast<float*>(ws + wl.total) : out;
        RT_CUDA(cudaMemsetAsync(master, 0, n_acc * sizeof(double), st));
        RT_CUDA(cudaMemsetAsync(scratch, 0, n_acc * sizeof(float), st));             // D14: overwrite
        const Batching bt = plan_batches(n_src, P.n_slots, pl.map_src);
        const int all_slots = P.n_slots;
        P.acc = scratch;
        long long db = ((long long)(n_acc / 4) + fin_threads - 1) / fin_threads;
        if (db > 148 * 16) db = 148 * 16;
        // two batches at a time, each into its own scratch grid; the second overlaps the tail of the first
        float* scratch2 = (step || pl.ktri) ? nullptr : reinterpret_cast<float*>(ws + wl.scratch2_at);
        if (scratch2) RT_CUDA(cudaMemsetAsync(scratch2, 0, n_acc * sizeof(float), st));
        const int sb = (n_src + bt.src_per_batch - 1) / bt.src_per_batch, db_n = (all_slots + bt.slots_per_batch - 1) / bt.slots_per_batch;
        auto select = [&](int b) {
            const int s0 = (b / db_n) * bt.src_per_batch, d0 = (b % db_n) * bt.slots_per_batch;
            P.src_begin = s0;
            P.n_src = std::min(bt.src_per_batch, n_src - s0);
            P.slot_begin = d0;
            P.n_slots = std::min(bt.slots_per_batch, all_slots - d0);
        };
        for (int b = 0; b < sb * db_n; b += scratch2 ? 2 : 1) {
            select(b);
            P.acc = scratch;
            const int rcb = launch_march<4, float>(P, true, st);
            if (rcb != RT_OK) return rcb;
            const bool pair = scratch2 && b + 1 < sb * db_n;
            if (pair) {
                select(b + 1);
                P.acc = scratch2;
                const int rcc = launch_march<4, float>(P, true, st, true);
                if (rcc != RT_OK) return rcc;
            }
            rt::drain_kernel<<<unsigned(db), fin_threads, 0, st>>>(master, scratch, pair ? scratch2 : nullptr, (long long)n_acc);
            RT_CUDA(cudaGetLastError());
        }
        if (step)
            rt::step_finalize_kernel<<<unsigned(fin_blocks), fin_threads, 0, st>>>(master, out, ck.cells, step->accumulate);
        else
            rt::snapshot_finalize_kernel<double><<<unsigned(fin_blocks), fin_threads, 0, st>>>(master, out, ck.cells, n_steps);
        RT_CUDA(cudaGetLastError());
        return RT_OK;
    }
    if (step) {                        // 1 bin per thread: fp64 reductions into the workspace grid, then the update of out
        P.acc = master;
        RT_CUDA(cudaMemsetAsync(master, 0, n_acc * sizeof(double), st));
        const int rcs = vec4 ? launch_march<4, double>(P, true, st) : launch_march<1, double>(P, true, st);
        if (rcs != RT_OK) return rcs;
        rt::step_finalize_kernel<<<unsigned(fin_blocks), fin_threads, 0, st>>>(master, out, ck.cells, step->accumulate);
        RT_CUDA(cudaGetLastError());
        return RT_OK;
    }

    // the accumulation grid: fp64 in the workspace (default), or `out` itself (RT_VARIANT_FLAG_ACC_F32)
    P.acc = pl.acc64 ? static_cast<void*>(master) : static_cast<void*>(out);
    if (pl.acc64 && pl.sliding && !vec4 && !pl.ktri) {       // the one-bin kernel spreads its reductions over copies
        P.acc_copies = wl.acc_copies;
        P.acc_copy_stride = (long long)n_acc;
    }
    RT_CUDA(cudaMemsetAsync(P.acc, 0, n_acc * (pl.acc64 ? sizeof(double) * size_t(P.acc_copies) : sizeof(float)), st));   // D14: overwrite
    int rc3;
    if (vec4) rc3 = pl.acc64 ? launch_march<4, double>(P, pl.sliding, st) : launch_march<4, float>(P, pl.sliding, st);
    else rc3 = pl.acc64 ? launch_march<1, double>(P, pl.sliding, st) : launch_march<1, float>(P, pl.sliding, st);
    if (rc3 != RT_OK) return rc3;
    if (pl.acc64) {
        rt::snapshot_finalize_kernel<double><<<unsigned(fin_blocks), fin_threads, 0, st>>>(master, out, ck.cells, n_steps,
                                                                                          P.acc_copies, P.acc_copy_stride);
        RT_CUDA(cudaGetLastError());
    } else if (n_steps > 1) {
        rt::snapshot_finalize_kernel<float><<<unsigned(fin_blocks), fin_threads, 0, st>>>(out, out, ck.cells, n_steps);
        RT_CUDA(cudaGetLastError());
    }
    return RT_OK;
}

}  // namespace

// rt_march_static: the workspace of callers that may not allocate (code under CUDA graph capture, serving loops,
// harnesses that forbid cudaMalloc).  A file-scope device array: every GPU that loads the library holds these
// RT_STATIC_WORKSPACE_BYTES until the process exits, every rt_march_static call on a device shares them.
// In host code the NAME of the array is a host-side stand-in, not a device address; the device address comes from
// cudaGetSymbolAddress, asked once per device with that device current.
static __device__ __align__(256) unsigned char g_static_workspace[RT_STATIC_WORKSPACE_BYTES];

namespace {

constexpr int kMaxStaticDevices = 64;
std::mutex g_static_mutex;
void* g_static_ptr[kMaxStaticDevices] = {};

// device address of g_static_workspace on the CURRENT device (no allocation: the array is part of the loaded module)
int static_workspace(void** ptr) {
    int dev = -1;
    RT_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxStaticDevices) return RT_EINVAL;
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[dev]) {
        void* p = nullptr;
        RT_CUDA(cudaGetSymbolAddress(&p, g_static_workspace));
        if (!p || (uintptr_t(p) & 255u)) return RT_EWORKSPACE;
        g_static_ptr[dev] = p;
    }
    *ptr = g_static_ptr[dev];
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

size_t rt_static_workspace_bytes(void) { return size_t(RT_STATIC_WORKSPACE_BYTES); }

int rt_march_static(const float* j, const float* kappa, int nx, int ny, int nz, const float* sources, int n_src, int n_rays,
                    int n_bins, float step_size, float c, float dt, int n_steps, float* out, void* stream) {
    // arguments and size first, on the host: a call that does not fit is refused before any CUDA call
    Checked ck;
    const int rc = check_args(j, kappa, nx, ny, nz, sources, n_src, n_rays, n_bins, step_size, c, dt, n_steps, out, &ck);
    if (rc != RT_OK) return rc;
    const size_t need = workspace_layout(nx, ny, nz, n_src, n_rays, n_steps, n_bins).total;
    if (need > size_t(RT_STATIC_WORKSPACE_BYTES)) return RT_ETOOBIG;
    void* ws = nullptr;
    const int rs = static_workspace(&ws);
    if (rs != RT_OK) return rs;
    // the march itself is rt_march's: it zeroes what it sums into (fp64 grid, fp32 scratch) and rebuilds the ray and
    // source orders on the stream in every call, so the contents the last call left in the array do not matter
    return march_impl(j, kappa, nx, ny, nz, sources, n_src, n_rays, n_bins, step_size, c, dt, n_steps, out, ws,
                      size_t(RT_STATIC_WORKSPACE_BYTES), stream, RT_VARIANT_DEFAULT);
}

int rt_march_trilinear_kappa(const float* j, const float* kappa, int nx, int ny, int nz, const float* sources, int n_src,
                             int n_rays, int n_bins, float step_size, float c, float dt, int n_steps, float* out,
                             void* workspace, size_t workspace_bytes, void* stream) {
    return march_impl(j, kappa, nx, ny, nz, sources, n_src, n_rays, n_bins, step_size, c, dt, n_steps, out, workspace,
                      workspace_bytes, stream, kVariantKappaTrilinear);
}

int rt_march_jvp_kappa(const float* j, const float* kappa, const float* dkappa, int nx, int ny, int nz, const float* sources,
                       int n_src, int n_rays, int n_bins, float step_size, float c, float dt, int n_steps, float* tangent,
                       void* workspace, size_t workspace_bytes, void* stream) {
    if (!dkappa) return RT_EINVAL;
    if (uintptr_t(dkappa) & 3u) return RT_EALIGN;
    if (!(step_size < 1.0f)) return RT_EINVAL;         // (argument order: the other checks are march_impl's)
    return march_impl(j, kappa, nx, ny, nz, sources, n_src, n_rays, n_bins, step_size, c, dt, n_steps, tangent, workspace,
                      workspace_bytes, stream, RT_VARIANT_DEFAULT, nullptr, dkappa);
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

size_t rt_adjoint_workspace_bytes(int nx, int ny, int nz, int n_src, int n_rays, int n_bins, int n_steps) {
    const size_t base = rt_workspace_bytes(nx, ny, nz, n_src, n_rays, n_bins, 1);
    if (!base || n_steps < 1) return 0;
    const size_t cells = size_t(nx) * ny * nz * n_bins;
    return align_up(base, 256) + (n_steps > 1 ? cells * size_t(n_steps) * sizeof(float) : 0);
}

int rt_march_adjoint_j(const float* gbar, const float* kappa, int nx, int ny, int nz, const float* sources, int n_src,
                       int n_rays, int n_bins, float step_size, float c, float dt, int n_steps, float* grad_j,
                       void* workspace, size_t workspace_bytes, void* stream) {
    Checked ck;
    const int rc = check_args(gbar, kappa, nx, ny, nz, sources, n_src, n_rays, n_bins, step_size, c, dt, n_steps,
                              grad_j, &ck);
    if (rc != RT_OK) return rc;
    const Workspace wl = workspace_layout(nx, ny, nz, n_src, n_rays, 1, n_bins);
    const size_t need = rt_adjoint_workspace_bytes(nx, ny, nz, n_src, n_rays, n_bins, n_steps);
    if (!workspace || workspace_bytes < need || (uintptr_t(workspace) & 15u)) return RT_EWORKSPACE;
    char* ws = static_cast<char*>(workspace);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const Plan pl = default_plan(n_src);
    rt::MarchParams P = base_params(nullptr, kappa, nx, ny, nz, sources, n_src, n_rays, n_bins, step_size, n_steps, ck, pl);
    const int rc2 = build_orders(P, pl, wl, ws, st);
    if (rc2 != RT_OK) return rc2;
    double* master = reinterpret_cast<double*>(ws + wl.acc_at);
    P.acc = master;
    RT_CUDA(cudaMemsetAsync(master, 0, size_t(ck.cells) * sizeof(double), st));
    const int threads = 256;
    long long blocks = (ck.cells + threads - 1) / threads;
    if (blocks > 148 * 16) blocks = 148 * 16;
    const float* gsuf = gbar;
    if (n_steps > 1) {                       // the snapshots are cumulative: step m feeds gbar[m], gbar[m+1], ...
        float* gs = reinterpret_cast<float*>(ws + align_up(wl.total, 256));
        rt::suffix_sum_kernel<<<unsigned(blocks), threads, 0, st>>>(gbar, gs, ck.cells, n_steps);
        RT_CUDA(cudaGetLastError());
        gsuf = gs;
    }
    const long long mb = rt::march_blocks(n_src, P.n_slots, P.n_groups, P.map_src);
    if (mb > 2147483647LL) return RT_EINVAL;
    if (n_bins == 1 && wl.brick_bytes && step_size < 1.0f) {
        // one bin: deposits as vector reductions into the fp32 brick scratch, drained into the fp64 grid during the march
        P.scratch = reinterpret_cast<float*>(ws + wl.brick_at);
        RT_CUDA(cudaMemsetAsync(P.scratch, 0, wl.brick_bytes, st));
        P.n_drain_units = std::max<long long>(1, (long long)(wl.brick_bytes / 16));
        const long long per = (P.n_drain_units * drain_rounds((long long)n_src * n_rays) + mb - 1) / mb;
        P.drain_units_per_block = std::min<long long>(std::max<long long>(per, 1), rt::kDrainMaxUnits);
        if (pl.map_src) rt::adjoint_kernel<6, false, true, true><<<unsigned(mb), rt::kThreads, 0, st>>>(P, gsuf, nullptr, 0);
        else rt::adjoint_kernel<6, false, true><<<unsigned(mb), rt::kThreads, 0, st>>>(P, gsuf, nullptr, 0);
        RT_CUDA(cudaGetLastError());
        rt::snapshot_finalize_scratch_kernel<true><<<unsigned(blocks), threads, 0, st>>>(master, P.scratch, grad_j, ck.cells, 1,
                                                                                        rt::brick_geom(nx, ny, nz), ny, nz, 1);
        RT_CUDA(cudaGetLastError());
        return RT_OK;
    }
    if (pl.map_src) rt::adjoint_kernel<6, false, false, true><<<unsigned(mb), rt::kThreads, 0, st>>>(P, gsuf, nullptr, 0);
    else rt::adjoint_kernel<6, false><<<unsigned(mb), rt::kThreads, 0, st>>>(P, gsuf, nullptr, 0);
    RT_CUDA(cudaGetLastError());
    rt::snapshot_finalize_kernel<double><<<unsigned(blocks), threads, 0, st>>>(master, grad_j, ck.cells, 1);
    RT_CUDA(cudaGetLastError());
    return RT_OK;
}

// rt_march_adjoint_kappa records I_{k+1} of every substep of every ray of a launch: 4 bytes per
// ray-substep-bin.  Sources are marched in batches so that this record stays below kForwardRecordLimit.
constexpr size_t kForwardRecordLimit = size_t(8) << 30;      // C2: 2 batches, 27.3 ms; 2 GiB (8 batches, 8 tails): 28.4 ms
struct KappaBatch {
    int src_per_batch;
    size_t record_bytes;
};
// record_limit: bytes the record of one batch may take (0 = kForwardRecordLimit; the _ex entries let tests force
// several batches on small cases); a batch is never smaller than one warp's worth of sources
KappaBatch plan_kappa_batches(int n_src, int n_slots, int n_groups, bool map_src, long long K, size_t record_limit) {
    if (!record_limit) record_limit = kForwardRecordLimit;
    const int unit = map_src ? 32 : 1;                               // sources come in whole warps' worth
    const int n_units = (n_src + unit - 1) / unit;
    auto bytes_for = [&](int n) {
        return size_t(rt::march_blocks(n, n_slots, n_groups, map_src ? 1 : 0)) * rt::kThreads * size_t(K) * sizeof(float);
    };
    int units = int(std::max<size_t>(1, record_limit / std::max<size_t>(1, bytes_for(unit))));
    units = std::min(units, n_units);
    KappaBatch kb;
    kb.src_per_batch = std::min(units * unit, map_src ? n_units * unit : n_src);
    kb.record_bytes = bytes_for(std::min(kb.src_per_batch, n_src));
    return kb;
}

size_t rt_adjoint_kappa_workspace_bytes_ex(int nx, int ny, int nz, int n_src, int n_rays, int n_bins, float step_size,
                                           float c, float dt, int n_steps, size_t record_limit) {
    const size_t base = rt_adjoint_workspace_bytes(nx, ny, nz, n_src, n_rays, n_bins, n_steps);
    if (!base || !positive_finite(step_size) || !positive_finite(c) || !positive_finite(dt)) return 0;
    const long long ns = substeps(step_size, c, dt);
    if (ns < 1 || ns * n_steps > 2147483647LL) return 0;
    const Plan pl = default_plan(n_src);
    return align_up(base, 256) +
           plan_kappa_batches(n_src, ray_slots(n_rays), n_bins, pl.map_src, ns * n_steps, record_limit).record_bytes;
}

size_t rt_adjoint_kappa_workspace_bytes(int nx, int ny, int nz, int n_src, int n_rays, int n_bins, float step_size,
                                        float c, float dt, int n_steps) {
    return rt_adjoint_kappa_workspace_bytes_ex(nx, ny, nz, n_src, n_rays, n_bins, step_size, c, dt, n_steps, 0);
}

int rt_march_adjoint_kappa(const float* gbar, const float* j, const float* kappa, int nx, int ny, int nz,
                           const float* sources, int n_src, int n_rays, int n_bins, float step_size, float c, float dt,
                           int n_steps, float* grad_kappa, void* workspace, size_t workspace_bytes, void* stream) {
    return rt_march_adjoint_kappa_ex(gbar, j, kappa, nx, ny, nz, sources, n_src, n_rays, n_bins, step_size, c, dt, n_steps,
                                     grad_kappa, workspace, workspace_bytes, stream, 0);
}

int rt_march_adjoint_kappa_ex(const float* gbar, const float* j, const float* kappa, int nx, int ny, int nz,
                              const float* sources, int n_src, int n_rays, int n_bins, float step_size, float c, float dt,
                              int n_steps, float* grad_kappa, void* workspace, size_t workspace_bytes, void* stream,
                              size_t record_limit) {
    if (!gbar) return RT_EINVAL;
    Checked ck;
    const int rc = check_args(j, kappa, nx, ny, nz, sources, n_src, n_rays, n_bins, step_size, c, dt, n_steps,
                              grad_kappa, &ck);
    if (rc != RT_OK) return rc;
    if (uintptr_t(gbar) & 3u) return RT_EALIGN;
    const Workspace wl = workspace_layout(nx, ny, nz, n_src, n_rays, 1, n_bins);
    const size_t base = rt_adjoint_workspace_bytes(nx, ny, nz, n_src, n_rays, n_bins, n_steps);
    const size_t need = rt_adjoint_kappa_workspace_bytes_ex(nx, ny, nz, n_src, n_rays, n_bins, step_size, c, dt, n_steps,
                                                            record_limit);
    if (!workspace || workspace_bytes < need || (uintptr_t(workspace) & 15u)) return RT_EWORKSPACE;
    char* ws = static_cast<char*>(workspace);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const Plan pl = default_plan(n_src);
    rt::MarchParams P = base_params(j, kappa, nx, ny, nz, sources, n_src, n_rays, n_bins, step_size, n_steps, ck, pl);
    const int rc2 = build_orders(P, pl, wl, ws, st);
    if (rc2 != RT_OK) return rc2;
    double* master = reinterpret_cast<double*>(ws + wl.acc_at);
    P.acc = master;
    RT_CUDA(cudaMemsetAsync(master, 0, size_t(ck.cells) * sizeof(double), st));
    const int threads = 256;
    long long blocks = (ck.cells + threads - 1) / threads;
    if (blocks > 148 * 16) blocks = 148 * 16;
    const float* gsuf = gbar;
    if (n_steps > 1) {
        float* gs = reinterpret_cast<float*>(ws + align_up(wl.total, 256));
        rt::suffix_sum_kernel<<<unsigned(blocks), threads, 0, st>>>(gbar, gs, ck.cells, n_steps);
        RT_CUDA(cudaGetLastError());
        gsuf = gs;
    }
    if (pl.map_src && step_size < 1.0f) {       // do the sources share their cell fractions? (rt_march_phased.cuh)
        int* flag = reinterpret_cast<int*>(ws + wl.flag_at);
        rt::same_fraction_kernel<<<1, 256, 0, st>>>(flag, sources, n_src, step_size);
        RT_CUDA(cudaGetLastError());
        P.same_frac = flag;
    }
    const long long K = ck.n_sub * n_steps;
    const KappaBatch kb = plan_kappa_batches(n_src, P.n_slots, P.n_groups, pl.map_src, K, record_limit);
    float* fwd = reinterpret_cast<float*>(ws + align_up(base, 256));
    for (int s0 = 0; s0 < n_src; s0 += kb.src_per_batch) {
        P.src_begin = s0;
        P.n_src = std::min(kb.src_per_batch, n_src - s0);
        const long long mb = rt::march_blocks(P.n_src, P.n_slots, P.n_groups, P.map_src);
        if (mb > 2147483647LL) return RT_EINVAL;
        const long long stride = mb * rt::kThreads;
        if (step_size < 1.0f) {        // the phased march, in its weight-table and its plain instantiation (one of them returns)
            P.record = fwd;
            P.record_stride = stride;
            if (pl.map_src) rt::march_phased_kernel<1, true, false, float, false, false, false, true><<<unsigned(mb), rt::kThreads, 0, st>>>(P);
            rt::march_phased_kernel<1, false, false, float, false, false, false, true><<<unsigned(mb), rt::kThreads, 0, st>>>(P);
        } else {
            rt::march_sliding_kernel<1, double, 8, false, false, true><<<unsigned(mb), rt::kThreads, 0, st>>>(P, fwd, stride);
        }
        RT_CUDA(cudaGetLastError());
        if (pl.map_src) rt::adjoint_kernel<4, true, false, true><<<unsigned(mb), rt::kThreads, 0, st>>>(P, gsuf, fwd, stride);
        else rt::adjoint_kernel<4, true><<<unsigned(mb), rt::kThreads, 0, st>>>(P, gsuf, fwd, stride);
        RT_CUDA(cudaGetLastError());
    }
    rt::snapshot_finalize_kernel<double><<<unsigned(blocks), threads, 0, st>>>(master, grad_kappa, ck.cells, 1);
    RT_CUDA(cudaGetLastError());
    return RT_OK;
}

size_t rt_state_bytes(int n_src, int n_rays, int n_bins) {
    if (n_src < 1 || n_rays < 1 || n_bins < 1) return 0;
    return size_t(2) * size_t(n_src) * size_t(n_rays) * size_t(n_bins) * sizeof(float);
}

int rt_state_reset(float* state, int n_src, int n_rays, int n_bins, void* stream) {
    if (!state || n_src < 1 || n_rays < 1 || n_bins < 1) return RT_EINVAL;
    const long long n = (long long)n_src * n_rays * n_bins;
    long long blocks = (n + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    rt::state_reset_kernel<<<unsigned(blocks), 256, 0, static_cast<cudaStream_t>(stream)>>>(state, state + n, n);
    RT_CUDA(cudaGetLastError());
    return RT_OK;
}

size_t rt_step_workspace_bytes(int nx, int ny, int nz, int n_src, int n_rays, int n_bins) {
    const size_t base = rt_workspace_bytes(nx, ny, nz, n_src, n_rays, n_bins, 1);
    return base ? base + step_scratch_bytes((long long)nx * ny * nz * n_bins, n_bins) : 0;
}

int rt_march_step(const float* j, const float* kappa, int nx, int ny, int nz, const float* sources, int n_src,
                  int n_rays, int n_bins, float step_size, float c, float dt, long long k_begin, float* state,
                  float* out, int accumulate, void* workspace, size_t workspace_bytes, void* stream) {
    const StepArgs sa{state, k_begin, accumulate};
    return march_impl(j, kappa, nx, ny, nz, sources, n_src, n_rays, n_bins, step_size, c, dt, 1, out, workspace,
                      workspace_bytes, stream, RT_VARIANT_DEFAULT, &sa);
}

// rt_march_host's device buffers come from a private stream-ordered memory pool per device that keeps what it has
// been given (release threshold = max), so repeated calls do not pay cudaMalloc/cudaFree; rt_host_release() trims it.
// rt_march_host holds g_pool_use shared for the whole call, rt_host_release takes it exclusively: a pool is never
// destroyed under a call that is using it.
static std::mutex g_pool_mutex;
static std::shared_mutex g_pool_use;
static cudaMemPool_t g_pools[64] = {};

static cudaError_t host_pool(cudaMemPool_t* pool) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_pool_mutex);
    if (!g_pools[dev]) {
        cudaMemPoolProps props = {};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        e = cudaMemPoolCreate(&g_pools[dev], &props);
        if (e != cudaSuccess) { g_pools[dev] = nullptr; return e; }
        unsigned long long keep = ~0ull;
        cudaMemPoolSetAttribute(g_pools[dev], cudaMemPoolAttrReleaseThreshold, &keep);
    }
    *pool = g_pools[dev];
    return cudaSuccess;
}

int rt_host_release(void) {
    std::unique_lock<std::shared_mutex> idle(g_pool_use);       // waits for running rt_march_host calls
    std::lock_guard<std::mutex> lock(g_pool_mutex);
    for (auto& p : g_pools)
        if (p) {
            cudaMemPoolDestroy(p);
            p = nullptr;
        }
    return RT_OK;
}

int rt_march_host(const float* j, const float* kappa, int nx, int ny, int nz, const float* sources, int n_src,
                  int n_rays, int n_bins, float step_size, float c, float dt, int n_steps, float* out) {
    Checked ck;
    const int rc = check_args(j, kappa, nx, ny, nz, sources, n_src, n_rays, n_bins, step_size, c, dt, n_steps, out, &ck);
    if (rc != RT_OK) return rc;
    const size_t grid_b = size_t(ck.cells) * sizeof(float), out_b = grid_b * size_t(n_steps);
    const size_t src_b = size_t(n_src) * 3 * sizeof(float);
    const size_t ws_b = rt_workspace_bytes(nx, ny, nz, n_src, n_rays, n_bins, n_steps);
    // one allocation: [j][kappa][out][workspace][sources], every part 256-byte aligned
    const size_t at_k = align_up(grid_b, 256), at_out = at_k + align_up(grid_b, 256), at_ws = at_out + align_up(out_b, 256),
                 at_src = at_ws + align_up(ws_b, 256), total = at_src + align_up(src_b, 256);
    char* base = nullptr;
    cudaMemPool_t pool = nullptr;
    cudaStream_t st = nullptr;
    int result = RT_OK;
    std::shared_lock<std::shared_mutex> in_use(g_pool_use);
    auto ok = [&](cudaError_t err, const char* where) {
        if (err != cudaSuccess && result == RT_OK) result = cuda_fail(err, where);
        return err == cudaSuccess;
    };
    if (ok(host_pool(&pool), "cudaMemPoolCreate") &&
        ok(cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking), "cudaStreamCreate") &&
        ok(cudaMallocFromPoolAsync(reinterpret_cast<void**>(&base), total, pool, st), "cudaMallocFromPoolAsync") &&
        ok(cudaMemcpyAsync(base, j, grid_b, cudaMemcpyHostToDevice, st), "H2D j") &&
        ok(cudaMemcpyAsync(base + at_k, kappa, grid_b, cudaMemcpyHostToDevice, st), "H2D kappa") &&
        ok(cudaMemcpyAsync(base + at_src, sources, src_b, cudaMemcpyHostToDevice, st), "H2D sources")) {
        result = march_impl(reinterpret_cast<float*>(base), reinterpret_cast<float*>(base + at_k), nx, ny, nz,
                            reinterpret_cast<float*>(base + at_src), n_src, n_rays, n_bins, step_size, c, dt, n_steps,
                            reinterpret_cast<float*>(base + at_out), base + at_ws, ws_b, st, RT_VARIANT_DEFAULT);
        if (result == RT_OK) ok(cudaMemcpyAsync(out, base + at_out, out_b, cudaMemcpyDeviceToHost, st), "D2H out");
    }
    if (base) cudaFreeAsync(base, st);
    if (st) {
        ok(cudaStreamSynchronize(st), "cudaStreamSynchronize");
        cudaStreamDestroy(st);
    }
    return result;
}

size_t rt_workspace_bytes(int nx, int ny, int nz, int n_src, int n_rays, int n_bins, int n_steps) {
    if (nx < 1 || ny < 1 || nz < 1 || n_src < 1 || n_rays < 1 || n_bins < 1 || n_steps < 1 || n_rays > (1 << 30))
        return 0;
    const long long cells = (long long)nx * ny;
    if (cells > 2147483647LL || cells * nz > 2147483647LL || cells * nz * n_bins > 2147483647LL) return 0;
    return workspace_layout(nx, ny, nz, n_src, n_rays, n_steps, n_bins).total;
}

int rt_substeps_per_step(float step_size, float c, float dt) {
    if (!positive_finite(step_size) || !positive_finite(c) || !positive_finite(dt)) return RT_EINVAL;
    const long long ns = substeps(step_size, c, dt);
    return ns < 1 ? RT_EINVAL : int(ns);
}

int rt_launch_count(int nx, int ny, int nz, int n_src, int n_rays, int n_bins, int n_steps) {
    if (nx < 1 || ny < 1 || nz < 1 || n_src < 1 || n_rays < 1 || n_bins < 1 || n_steps < 1) return RT_EINVAL;
    const Plan pl = default_plan(n_src);
    // key, scan, scatter, march, snapshots; not drained (bins in fours, few deposits per element): + state reset, two marches
    if (workspace_layout(nx, ny, nz, n_src, n_rays, n_steps, n_bins).sort_bytes) return n_bins % 4 == 0 ? 7 : 5;
    const int setup = 1 + ((pl.map_src && n_src <= kMaxSortedSources) ? 1 : 0);     // ray order, (source order)
    // the phased march (what rt_march runs when substeps are shorter than a cell): (fraction test, the weight-table
    // instantiation,) the plain instantiation -- one of the two returns at once --, snapshots
    return setup + (pl.map_src ? 2 : 0) + 2;
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
    P.j = j; P.kappa = kappa; P.sources = source_pos; P.acc = nullptr; P.ray_order = nullptr; P.src_order = nullptr; P.map_src = 0;
    P.nx = nx; P.ny = ny; P.nz = nz; P.nb = n_bins;
    P.n_src = 1; P.src_begin = 0; P.slot_begin = 0; P.n_rays = n_rays; P.n_slots = n_rays; P.n_groups = 1; P.n_steps = 1; P.n_sub = n_sub;
    P.ds = double(step_size); P.ds_f = step_size; P.emis = step_size; P.att_scale = 0.0f; P.snap_stride = 0;
    P.state_I = nullptr; P.state_T = nullptr; P.k0 = 0; P.kappa_trilinear = 0;
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

int rt_bench_red_ceiling(int mode, void* grid, int nx, int ny, int nz, int n_bins, long long n_red, unsigned int seed,
                         long long* n_issued, void* stream) {
    if (!grid || mode < 0 || mode > 9 || nx < 2 || ny < 2 || nz < 2 || n_bins < 1 || n_red < 1) return RT_EINVAL;
    const long long elems = (long long)nx * ny * nz * n_bins;
    if (elems > 2147483647LL || elems < 32) return RT_EINVAL;
    const bool vec = (n_bins % 4 == 0) && !(uintptr_t(grid) & 15u);
    if (mode == 1 && (elems % 4 || (uintptr_t(grid) & 15u))) return RT_EALIGN;
    if ((mode == 6 || mode == 7) && (uintptr_t(grid) & 7u)) return RT_EALIGN;
    const int threads = 256, blocks = 148 * 8;
    // reductions (red instructions x lanes) one thread issues per iteration
    long long per_iter = 8LL;
    if (mode == 2 || mode == 5) per_iter = 8LL * (vec ? n_bins / 4 : n_bins);
    if (mode == 7) per_iter = 8LL * n_bins;
    const long long lanes = (long long)threads * blocks;
    long long iters = (n_red + lanes * per_iter - 1) / (lanes * per_iter);
    if (iters > 2147483647LL) return RT_EINVAL;
    rt::CeilingParams P{static_cast<float*>(grid), nx, ny, nz, n_bins, int(iters), seed};
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
        case 6: rt::red_ceiling_kernel<6, 1><<<blocks, threads, 0, st>>>(P); break;
        case 7: rt::red_ceiling_kernel<7, 1><<<blocks, threads, 0, st>>>(P); break;
        case 8: rt::red_ceiling_kernel<8, 1><<<blocks, threads, 0, st>>>(P); break;
        case 9: rt::red_ceiling_kernel<9, 1><<<blocks, threads, 0, st>>>(P); break;
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
        case RT_ETOOBIG: return "the call needs more scratch than rt_march_static's static workspace holds (rt_static_workspace_bytes()); use rt_march with a workspace of rt_workspace_bytes()";
        default: return "unknown rtmarch error code";
    }
}

const char* rt_version(void) { return "rtmarch 0.8 (sm_100a; sliding-stencil march in warp-uniform phases, weight table per warp for sources sharing their cell fractions, fp32 scratch (window bricks / bin vectors) with vector reductions drained concurrently into an fp64 grid, rays sorted by tile on grids beyond the L2)"; }

}  // extern "C"
