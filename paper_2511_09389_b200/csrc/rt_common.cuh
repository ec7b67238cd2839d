// rt_common.cuh — shared device code of the ray-march kernels (sm_100a): launch parameters, the direction
// lattice, the 96-bit fixed-point position, bin-vector loads / reductions, and the thread -> ray mapping.
//
// Geometry is exact integer arithmetic (DESIGN.md §4 D3): a position is a 96-bit fixed-point number per axis
// (int32 cell, 64 fractional bits), x_k = (floor(x_0 2^64) + k floor(fl(ds n) 2^64)) / 2^64, advanced with an
// add-with-carry chain; floor(x_k) is the top word and the trilinear fraction is the next 32 bits.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace rt {

struct MarchParams {
    const float* j;
    const float* kappa;
    const float* dkappa;         // rt_march_jvp_kappa: the direction kappa is perturbed in (same layout), else nullptr
    const float* sources;        // [n_src][3]
    void* acc;                   // accumulation grid [n_steps][nx][ny][nz][nb], float or double: per-step INCREMENTS
    const uint32_t* ray_order;   // [n_slots] slot -> lattice index (0xFFFFFFFF = padding) or nullptr = identity
    const uint32_t* src_order;   // [n_src] rank -> source index (spatially sorted) or nullptr = identity
    int nx, ny, nz, nb;
    int n_src, n_rays, n_slots;  // n_src: sources of THIS launch, ranks src_begin .. src_begin + n_src - 1
    int src_begin;
    int slot_begin;              // direction slots of THIS launch: slot_begin .. slot_begin + n_slots - 1
    int n_groups;                // bin groups per ray (nb / NB)
    int n_steps, n_sub;          // time steps, substeps per step (N_s)
    int kappa_trilinear;         // reading D18 instead of D4 (rt_march_trilinear_kappa)
    int map_src;                 // 0: the lanes of a warp are 32 directions of one source; 1: 32 sources, one direction;
                                 // 2: consecutive entries of `perm` (rt_chunk.cuh: rays sorted by where they are)
    const uint32_t* perm;        // map_src = 2: [n_perm] entry = source * n_rays + lattice index
    long long n_perm;
    double ds;                   // step_size as double
    float ds_f;                  // step_size
    float emis;                  // ds * 4 pi / N_Omega: emission quadrature weight times solid-angle weight (D8)
    float att_scale;             // -ds * log2(e): exp(-kappa ds) = 2^(kappa * att_scale)
    long long snap_stride;       // elements per snapshot
    float* state_I;              // rt_march_step: carried I per (source, lattice index, bin), else nullptr
    float* state_T;              //                carried exp(-tau), same layout
    long long k0;                // substep index of the first substep of this launch (0 for rt_march)
    int first_left;              // state_I != nullptr: substeps left in the time step the launch starts in (0 = all n_sub); the
                                 // launch marches first_left + (n_steps - 1) n_sub substeps
    const int* same_frac;        // device flag, or nullptr: all sources share their cell fractions -> the TABLE instantiation
                                 // of march_phased_kernel marches the call and the plain one returns at once (and vice versa)
    // march_sliding_kernel<..., COPIES = true>, else 1 / 0:
    int acc_copies;              // block b reduces into copy b % acc_copies of the accumulation grid ...
    long long acc_copy_stride;   // ... copies being acc_copy_stride elements apart (hot voxels meet fewer reductions)
    // march_phased_kernel: the fp32 scratch its rays deposit into (rt_brick.cuh: window bricks [n_steps][nx][ny+1][nz+1][4]
    // for one bin per thread, the plain grid [n_steps][nx][ny][nz][nb] for four), drained into the fp64 grid `acc`
    // while the march runs
    float* scratch;
    // march_phased_kernel<..., RECORD> (rt_march_adjoint_kappa): nothing is deposited; I_{k+1} (x 4 pi/N_Omega) of substep k
    // goes to record[k * record_stride + thread]
    float* record;
    long long record_stride;
    long long drain_units_per_block;   // 16-byte units of the scratch one block drains when its rays are done
    long long n_drain_units;           // 16-byte units of the whole scratch
};

constexpr uint32_t kPad = 0xFFFFFFFFu;
constexpr int kThreads = 128;    // threads per march block (4 warps)

// (3 - sqrt 5)/2 * 2^128, floored: the golden angle as a fraction of a turn in 0.128 fixed point
constexpr uint64_t kGoldenTurnHi = 0x61C8864680B583EAull;
constexpr uint64_t kGoldenTurnLo = 0x0C633F9FA31237CBull;

// i * golden turn mod 1 as a 0.64 fraction (error < 2^-64 + i 2^-128 turn)
__device__ __forceinline__ uint64_t golden_turn64(uint32_t i) {
    return uint64_t(i) * kGoldenTurnHi + __umul64hi(uint64_t(i), kGoldenTurnLo);
}

// ---------------------------------------------------------------------------------------------------
// direction lattice (D1): z_i = 1 - (2i+1)/N = (N-2i-1)/N, phi_i = i * pi (3 - sqrt 5).
// z and sqrt(1-z^2) use only correctly rounded IEEE double operations on exact integers (one division for z;
// (2i+1)/N, (2(N-i)-1)/N, their product and its square root for the radius), so the oracle, which states
// the same operations, gets bit-identical values; the azimuth is reduced exactly in integer arithmetic.
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ void fib_direction(uint32_t i, uint32_t n, double nh[3]) {
    const double q = (2.0 * double(i) + 1.0) / double(n);          // 1 - z
    const double q2 = (2.0 * double(n - i) - 1.0) / double(n);     // 1 + z
    const double z = (double(n) - 2.0 * double(i) - 1.0) / double(n);
    const int64_t t = int64_t(golden_turn64(i));                   // phi/(2 pi) mod 1 as a signed 0.64 fraction
    const double turn = double(t) * 5.42101086242752217e-20;       // * 2^-64  -> [-0.5, 0.5)
    double s, c;
    sincospi(2.0 * turn, &s, &c);
    const double r = sqrt(__dmul_rn(q, q2));                       // sqrt((1-z)(1+z))
    nh[0] = __dmul_rn(r, c);
    nh[1] = __dmul_rn(r, s);
    nh[2] = z;
}

// ---------------------------------------------------------------------------------------------------
// 96-bit fixed point: value = c + fh 2^-32 + fl 2^-64
// ---------------------------------------------------------------------------------------------------
struct Fx96 {
    int32_t c;
    uint32_t fh, fl;
};

// floor(v * 2^64) EXACTLY, for |v| < 2^30 (no floating-point rounding: the double's significand is shifted).
// mode kFxNegate returns -floor(v 2^64), mode kFxComplement returns -floor(v 2^64) - 1 (both exact): the
// increment and the position of a descending axis in travel coordinates (rt_march_sliding.cuh)
constexpr int kFxPlain = 0, kFxNegate = 1, kFxComplement = 2;

__device__ __forceinline__ Fx96 fx_from_double(double v, int mode = kFxPlain) {
    const long long bits = __double_as_longlong(v);
    const int e = int((bits >> 52) & 0x7FF);
    long long m = bits & 0xFFFFFFFFFFFFFll;
    if (e) m |= 1ll << 52;                                   // v = +-m 2^(e' - 1075), e' = max(e, 1)
    if (bits < 0) m = -m;
    const int sh = (e ? e : 1) - 1011;                       // v 2^64 = m 2^sh; sh <= 41 since |v| < 2^30
    __int128 n;
    if (sh >= 0) n = __int128(m) << sh;
    else if (sh > -64) n = __int128(m >> (-sh));             // arithmetic shift = floor
    else n = (m < 0) ? -1 : 0;
    if (mode == kFxNegate) n = -n;
    if (mode == kFxComplement) n = ~n;
    Fx96 r;
    r.c = int32_t(int64_t(n >> 64));
    r.fh = uint32_t(uint64_t(n) >> 32);
    r.fl = uint32_t(uint64_t(n));
    return r;
}

__device__ __forceinline__ void fx_add(Fx96& p, const Fx96& d) {
    asm("add.cc.u32 %0, %0, %3;\n\t"
        "addc.cc.u32 %1, %1, %4;\n\t"
        "addc.s32 %2, %2, %5;"
        : "+r"(p.fl), "+r"(p.fh), "+r"(p.c)
        : "r"(d.fl), "r"(d.fh), "r"(d.c));
}

__device__ __forceinline__ void fx_sub(Fx96& p, const Fx96& d) {
    asm("sub.cc.u32 %0, %0, %3;\n\t"
        "subc.cc.u32 %1, %1, %4;\n\t"
        "subc.s32 %2, %2, %5;"
        : "+r"(p.fl), "+r"(p.fh), "+r"(p.c)
        : "r"(d.fl), "r"(d.fh), "r"(d.c));
}

// p += k d, exact (k >= 0, the product stays far below 2^127: paths are limited to 2^28 cells)
__device__ __forceinline__ void fx_advance(Fx96& p, const Fx96& d, long long k) {
    const __int128 pp = (__int128(p.c) << 64) | (__int128(p.fh) << 32) | __int128(p.fl);
    const __int128 dd = (__int128(d.c) << 64) | (__int128(d.fh) << 32) | __int128(d.fl);
    const __int128 n = pp + dd * __int128(k);
    p.c = int32_t(int64_t(n >> 64));
    p.fh = uint32_t(uint64_t(n) >> 32);
    p.fl = uint32_t(uint64_t(n));
}

// source coordinate a of source s, saturated to +-2^29 cells (rtmarch.h)
__device__ __forceinline__ double source_coord(const MarchParams& P, int s, int a) {
    const float x0 = __ldg(P.sources + 3 * size_t(s) + a);
    return double(fminf(fmaxf(x0, -536870912.0f), 536870912.0f));
}

// ---------------------------------------------------------------------------------------------------
// NB-wide (1 or 4 bins) loads and reductions into a float or a double accumulation grid
// ---------------------------------------------------------------------------------------------------
template <int NB> struct BinVec { float v[NB]; };

template <int NB> __device__ __forceinline__ BinVec<NB> ld_bins(const float* p);
template <> __device__ __forceinline__ BinVec<1> ld_bins<1>(const float* p) {
    BinVec<1> r;
    r.v[0] = __ldg(p);
    return r;
}
template <> __device__ __forceinline__ BinVec<4> ld_bins<4>(const float* p) {
    const float4 t = __ldg(reinterpret_cast<const float4*>(p));
    BinVec<4> r;
    r.v[0] = t.x; r.v[1] = t.y; r.v[2] = t.z; r.v[3] = t.w;
    return r;
}

__device__ __forceinline__ void red_bins(float* p, const BinVec<1>& a) {
    asm volatile("red.global.add.f32 [%0], %1;" ::"l"(p), "f"(a.v[0]) : "memory");
}
__device__ __forceinline__ void red_bins(float* p, const BinVec<4>& a) {
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(a.v[0]), "f"(a.v[1]), "f"(a.v[2]),
                 "f"(a.v[3])
                 : "memory");
}
template <int NB> __device__ __forceinline__ void red_bins(double* p, const BinVec<NB>& a) {
#pragma unroll
    for (int b = 0; b < NB; ++b)
        asm volatile("red.global.add.f64 [%0], %1;" ::"l"(p + b), "d"(double(a.v[b])) : "memory");
}

template <int NB> __device__ __forceinline__ bool any_nonzero(const BinVec<NB>& a) {
    bool nz = false;
#pragma unroll
    for (int b = 0; b < NB; ++b) nz |= (a.v[b] != 0.0f);
    return nz;
}

// ---------------------------------------------------------------------------------------------------
// thread -> (source, lattice index, bin group).  The bin group is the FASTEST lane index: the G = n_bins / NB
// threads that march the same ray for different bins sit in adjacent lanes, so their loads and reductions hit
// adjacent words of the bin-innermost grids (one 32-byte sector for 4 fp64 or 8 fp32 bins).  Two mappings of
// the rays:
//   map_src = 0  block = 128 consecutive (direction slot, group) pairs of one source (a patch of the sphere);
//   map_src = 1  block = 4 consecutive direction slots; each warp 32 consecutive (source, group) pairs of the
//                spatially sorted source list, ONE direction.  Rays of a warp are parallel; when the sources
//                share their fractional cell offsets (cell-centred sources) the lanes cross cell
//                faces in the same substep, so the stencil-slide branches are warp-uniform.
// Block order: direction chunk fastest, then source (chunk).
// ---------------------------------------------------------------------------------------------------
struct RayId {
    int src, group;
    uint32_t index;   // lattice index
};

__host__ __device__ inline long long perm_blocks(long long n_perm, int n_groups) {
    return (n_perm * n_groups + kThreads - 1) / kThreads;
}

__host__ __device__ inline long long march_blocks(int n_src, int n_slots, int n_groups, int map_src) {
    if (map_src) return (long long)((n_slots + 3) / 4) * (((long long)n_src * n_groups + 31) / 32);
    return (((long long)n_slots * n_groups + kThreads - 1) / kThreads) * n_src;
}

__device__ __forceinline__ bool ray_id(const MarchParams& P, RayId& id) {
    const uint32_t G = uint32_t(P.n_groups);
    uint32_t b = blockIdx.x, slot, s;
    if (P.map_src == 2) {
        const long long f = (long long)b * kThreads + threadIdx.x;       // (entry, group), group fastest
        const long long r = f / G;
        id.group = int(f - r * G);
        if (r >= P.n_perm) return false;
        const uint32_t e = __ldg(P.perm + r);
        id.src = int(e / uint32_t(P.n_rays));
        id.index = e - uint32_t(id.src) * uint32_t(P.n_rays);
        return true;
    }
    if (P.map_src) {
        const uint32_t chunks = (uint32_t(P.n_slots) + 3u) / 4u;
        slot = (b % chunks) * 4u + (threadIdx.x >> 5);
        const uint32_t f = (b / chunks) * 32u + (threadIdx.x & 31u);      // (source rank, group), group fastest
        s = f / G;
        id.group = int(f - s * G);
    } else {
        const uint32_t chunks = (uint32_t(P.n_slots) * G + kThreads - 1) / kThreads;
        const uint32_t f = (b % chunks) * kThreads + threadIdx.x;         // (direction slot, group), group fastest
        slot = f / G;
        id.group = int(f - slot * G);
        s = b / chunks;
    }
    if (slot >= uint32_t(P.n_slots) || s >= uint32_t(P.n_src)) return false;
    s += uint32_t(P.src_begin);
    slot += uint32_t(P.slot_begin);
    id.src = int(P.src_order ? P.src_order[s] : s);
    id.index = P.ray_order ? P.ray_order[slot] : slot;
    return id.index != kPad && id.index < uint32_t(P.n_rays);
}

}  // namespace rt
