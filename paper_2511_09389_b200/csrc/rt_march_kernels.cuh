// rt_march_kernels.cuh — the ray-march kernels (sm_100a).  One thread marches one (source, direction,
// bin-group) ray for all n_steps * N_s substeps of eq. (2) and issues its deposits
// as fp32 reductions (RED.E.ADD.F32 / RED.E.ADD.F32x4) into the one shared output grid.
//
// Geometry is exact integer arithmetic: the position is a 96-bit fixed-point number per axis (int32
// cell, 64 fractional bits) advanced by x_{k+1} = x_k + n ds with an add-with-carry chain,
// so x_k = x_0 + k (ds n) holds to 2^-64 cell per step with no drift, floor(x_k) is the top word and the
// trilinear fraction is the next 32 bits.  (DESIGN.md §7 explains why fp32 positions cannot meet the
// parity bar and why this is cheaper than fp64.)
//
// Two deposit strategies, same field:
//   direct  : 8 reductions per ray-substep, as the update rule is written;
//   sliding : the 8 stencil voxels are accumulated in registers and a voxel is reduced to memory only when
//             the ray's clamped stencil slides off it.  Accumulators and the cached j corners are indexed
//             trailing/leading along the ray's direction of travel, so a slide by one cell in one axis
//             flushes the 4 trailing voxels, moves 4, and loads 4 new j values.  Where an axis is clamped
//             (both indices equal: the ray is outside the box in that axis) the two slots are
//             merged, exact-zero accumulators are skipped, and a ray outside in all three axes issues one
//             reduction for the whole rest of its path.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace rt {

struct MarchParams {
    const float* j;
    const float* kappa;
    const float* sources;        // [n_src][3]
    float* out;                  // [n_steps][nx][ny][nz][nb]; holds per-step INCREMENTS until the prefix kernel runs
    const uint32_t* ray_order;   // [n_slots] slot -> lattice index (0xFFFFFFFF = padding) or nullptr = identity
    int nx, ny, nz, nb;
    int n_src, n_rays, n_slots;
    int n_groups;                // bin groups per ray (nb / NB)
    int n_steps, n_sub;          // time steps, substeps per step (N_s)
    double ds;                   // step_size as double
    float ds_f;                  // step_size
    float emis;                  // ds * 4 pi / N_Omega: emission quadrature weight times solid-angle weight (D8)
    long long snap_stride;       // elements per snapshot
};

constexpr uint32_t kPad = 0xFFFFFFFFu;
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
// 96-bit fixed point: value = c + fh 2^-32 + fl 2^-64 (D3: positions live on the 2^-64 cell grid)
// ---------------------------------------------------------------------------------------------------
struct Fx96 {
    int32_t c;
    uint32_t fh, fl;
};

// floor(v * 2^64) EXACTLY, for |v| < 2^30 (no floating-point rounding: the double's significand is shifted)
__device__ __forceinline__ Fx96 fx_from_double(double v) {
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

// ---------------------------------------------------------------------------------------------------
// NB-wide (1 or 4 bins) loads and reductions
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

template <int NB> __device__ __forceinline__ void red_bins(float* p, const BinVec<NB>& a);
template <> __device__ __forceinline__ void red_bins<1>(float* p, const BinVec<1>& a) {
    asm volatile("red.global.add.f32 [%0], %1;" ::"l"(p), "f"(a.v[0]) : "memory");
}
template <> __device__ __forceinline__ void red_bins<4>(float* p, const BinVec<4>& a) {
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(a.v[0]), "f"(a.v[1]), "f"(a.v[2]),
                 "f"(a.v[3])
                 : "memory");
}

template <int NB> __device__ __forceinline__ bool any_nonzero(const BinVec<NB>& a) {
    bool nz = false;
#pragma unroll
    for (int b = 0; b < NB; ++b) nz |= (a.v[b] != 0.0f);
    return nz;
}

// ---------------------------------------------------------------------------------------------------
// per-axis clamped stencil (D5): lo = clamp(floor x), hi = clamp(floor x + 1),
// weights (1-f, f) from the unclamped fraction.
// ---------------------------------------------------------------------------------------------------
struct AxisLoHi {
    int lo, hi;     // clamped indices
    float f, g;     // fraction in [0, 1] and its complement 1 - f, EACH rounded from the exact 32-bit fraction
};                  // (1.0f - f would carry f's absolute rounding error, 3e-8, into weights as small as 1e-5)

__device__ __forceinline__ AxisLoHi axis_lohi(const Fx96& p, int nmax) {
    AxisLoHi s;
    s.f = __uint2float_rn(p.fh) * 2.3283064365386963e-10f;    // 2^-32
    s.g = p.fh ? __uint2float_rn(0u - p.fh) * 2.3283064365386963e-10f : 1.0f;
    s.lo = min(max(p.c, 0), nmax);
    s.hi = min(max(p.c + 1, 0), nmax);
    return s;
}

// the same stencil in travel order: trailing (t) / leading (l) element offsets and weights
struct AxisTL {
    int t, l;
    float wt, wl;
};

__device__ __forceinline__ AxisTL axis_tl(const Fx96& p, int nmax, int stride, bool neg) {
    const AxisLoHi s = axis_lohi(p, nmax);
    const float g = s.g;
    AxisTL r;
    r.t = (neg ? s.hi : s.lo) * stride;
    r.l = (neg ? s.lo : s.hi) * stride;
    r.wt = neg ? s.f : g;
    r.wl = neg ? g : s.f;
    if (s.lo == s.hi) {        // clamped axis: both slots are the same voxel -> merge them (weights sum to 1)
        r.wt = 1.0f;
        r.wl = 0.0f;
    }
    return r;
}

// thread -> (source, ray slot, bin group); false if this thread has no ray
struct RayId {
    int src, group;
    uint32_t index;   // lattice index
};

__device__ __forceinline__ bool ray_id(const MarchParams& P, RayId& id) {
    // block order: slot chunk fastest, then bin group, then source, so neighbouring blocks share cache lines
    const uint32_t chunks = (uint32_t(P.n_slots) + blockDim.x - 1) / blockDim.x;
    uint32_t b = blockIdx.x;
    const uint32_t chunk = b % chunks;
    b /= chunks;
    id.group = int(b % uint32_t(P.n_groups));
    id.src = int(b / uint32_t(P.n_groups));
    const uint32_t slot = chunk * blockDim.x + threadIdx.x;
    if (slot >= uint32_t(P.n_slots)) return false;
    id.index = P.ray_order ? P.ray_order[slot] : slot;
    return id.index != kPad && id.index < uint32_t(P.n_rays);
}

struct RaySetup {
    Fx96 p[3], d[3];
    bool neg[3];
};

__device__ __forceinline__ RaySetup ray_setup(const MarchParams& P, const RayId& id) {
    RaySetup r;
    double nh[3];
    fib_direction(id.index, uint32_t(P.n_rays), nh);
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        float x0 = __ldg(P.sources + 3 * size_t(id.src) + a);
        x0 = fminf(fmaxf(x0, -536870912.0f), 536870912.0f);       // saturate to +-2^29 cells (rtmarch.h)
        r.p[a] = fx_from_double(double(x0));
        r.d[a] = fx_from_double(__dmul_rn(P.ds, nh[a]));
        r.neg[a] = nh[a] < 0.0;
    }
    return r;
}

// ===================================================================================================
// direct kernel: eq. (2) and the deposit exactly as written, 8 loads of j, 1 of kappa, 8 reductions
// ===================================================================================================
template <int NB>
__global__ void __launch_bounds__(128) march_direct_kernel(const MarchParams P) {
    RayId id;
    if (!ray_id(P, id)) return;
    RaySetup R = ray_setup(P, id);
    const int sx = P.ny * P.nz * P.nb, sy = P.nz * P.nb, sz = P.nb;
    const float* jg = P.j + id.group * NB;
    const float* kg = P.kappa + id.group * NB;
    float* og = P.out + id.group * NB;
    float I[NB], T[NB];     // I scaled by 4 pi/N_Omega; T = exp(-tau)
#pragma unroll
    for (int b = 0; b < NB; ++b) { I[b] = 0.0f; T[b] = 1.0f; }

    for (int m = 0; m < P.n_steps; ++m) {
        for (int k = 0; k < P.n_sub; ++k) {
            const AxisLoHi ax = axis_lohi(R.p[0], P.nx - 1), ay = axis_lohi(R.p[1], P.ny - 1),
                           az = axis_lohi(R.p[2], P.nz - 1);
            const int ox[2] = {ax.lo * sx, ax.hi * sx}, oy[2] = {ay.lo * sy, ay.hi * sy},
                      oz[2] = {az.lo * sz, az.hi * sz};
            const float wx[2] = {ax.g, ax.f}, wy[2] = {ay.g, ay.f}, wz[2] = {az.g, az.f};
            const BinVec<NB> kap = ld_bins<NB>(kg + ox[0] + oy[0] + oz[0]);
            float jv[NB];
#pragma unroll
            for (int b = 0; b < NB; ++b) jv[b] = 0.0f;
            float w[8];
            int off[8];
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                off[c] = ox[c >> 2] + oy[(c >> 1) & 1] + oz[c & 1];
                w[c] = wx[c >> 2] * wy[(c >> 1) & 1] * wz[c & 1];
                const BinVec<NB> jc = ld_bins<NB>(jg + off[c]);
#pragma unroll
                for (int b = 0; b < NB; ++b) jv[b] = fmaf(w[c], jc.v[b], jv[b]);
            }
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                const float a = expf(-kap.v[b] * P.ds_f);
                I[b] = fmaf(I[b], a, jv[b] * T[b] * P.emis);
                T[b] *= a;
            }
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                BinVec<NB> d;
#pragma unroll
                for (int b = 0; b < NB; ++b) d.v[b] = w[c] * I[b];
                red_bins<NB>(og + off[c], d);
            }
#pragma unroll
            for (int a = 0; a < 3; ++a) fx_add(R.p[a], R.d[a]);
        }
        og += P.snap_stride;
    }
}

// ===================================================================================================
// trace kernel (TEST HOOK): one thread marches one ray with the direct kernel's arithmetic and records, per
// substep, the position x_k (as double: cell + 64-bit fraction), I_{k+1} (UNscaled by 4 pi/N_Omega: emis = ds)
// and T_{k+1} = exp(-tau_{k+1}) for every bin.  No deposits.
// ===================================================================================================
__global__ void trace_ray_kernel(const MarchParams P, uint32_t ray_index, int n_sub, double* pos, float* trI, float* trT) {
    if (blockIdx.x || threadIdx.x) return;
    RayId id;
    id.src = 0; id.group = 0; id.index = ray_index;
    RaySetup R = ray_setup(P, id);
    const int sx = P.ny * P.nz * P.nb, sy = P.nz * P.nb, sz = P.nb;
    for (int b = 0; b < P.nb; ++b) {
        Fx96 p[3] = {R.p[0], R.p[1], R.p[2]};
        float I = 0.0f, T = 1.0f;
        for (int k = 0; k < n_sub; ++k) {
            const AxisLoHi ax = axis_lohi(p[0], P.nx - 1), ay = axis_lohi(p[1], P.ny - 1), az = axis_lohi(p[2], P.nz - 1);
            const int ox[2] = {ax.lo * sx, ax.hi * sx}, oy[2] = {ay.lo * sy, ay.hi * sy}, oz[2] = {az.lo * sz, az.hi * sz};
            const float wx[2] = {ax.g, ax.f}, wy[2] = {ay.g, ay.f}, wz[2] = {az.g, az.f};
            const float kap = __ldg(P.kappa + ox[0] + oy[0] + oz[0] + b);
            float jv = 0.0f;
            for (int c = 0; c < 8; ++c) {
                const float w = wx[c >> 2] * wy[(c >> 1) & 1] * wz[c & 1];
                jv = fmaf(w, __ldg(P.j + ox[c >> 2] + oy[(c >> 1) & 1] + oz[c & 1] + b), jv);
            }
            const float a = expf(-kap * P.ds_f);
            I = fmaf(I, a, jv * T * P.ds_f);
            T *= a;
            if (b == 0)
                for (int q = 0; q < 3; ++q)
                    pos[3 * size_t(k) + q] = double(p[q].c) + double(p[q].fh) * 2.3283064365386963e-10 +
                                             double(p[q].fl) * 5.42101086242752217e-20;
            trI[size_t(k) * P.nb + b] = I;
            trT[size_t(k) * P.nb + b] = T;
            for (int q = 0; q < 3; ++q) fx_add(p[q], R.d[q]);
        }
    }
}

// ===================================================================================================
// sliding-stencil kernel
// ===================================================================================================
// accumulator / j-cache slot for (plane p of axis AX, other two axes u, v); slots are [x][y][z] in travel order
template <int AX> __device__ __forceinline__ constexpr int slot(int p, int u, int v) {
    return AX == 0 ? (p * 4 + u * 2 + v) : (AX == 1 ? (u * 4 + p * 2 + v) : (u * 4 + v * 2 + p));
}

template <int NB> struct Sliding {
    BinVec<NB> acc[8];   // pending deposits for the 8 stencil voxels
    BinVec<NB> jc[8];    // j at the 8 stencil voxels
    int o[3][2];         // element offsets of the trailing/leading index per axis

    __device__ __forceinline__ int off(int s) const { return o[0][(s >> 2) & 1] + o[1][(s >> 1) & 1] + o[2][s & 1]; }

    __device__ __forceinline__ void flush_slot(float* og, int s) {
        if (any_nonzero<NB>(acc[s])) red_bins<NB>(og + off(s), acc[s]);
    }

    __device__ __forceinline__ void flush_all(float* og) {
#pragma unroll
        for (int s = 0; s < 8; ++s) {
            flush_slot(og, s);
#pragma unroll
            for (int b = 0; b < NB; ++b) acc[s].v[b] = 0.0f;
        }
    }

    __device__ __forceinline__ void load_all(const float* jg) {
#pragma unroll
        for (int s = 0; s < 8; ++s) jc[s] = ld_bins<NB>(jg + off(s));
    }

    // the stencil moved by one cell along AX: the old leading index is the new trailing index
    template <int AX> __device__ __forceinline__ void shift(float* og, const float* jg, int new_leading) {
#pragma unroll
        for (int u = 0; u < 2; ++u)
#pragma unroll
            for (int v = 0; v < 2; ++v) {
                const int s0 = slot<AX>(0, u, v), s1 = slot<AX>(1, u, v);
                flush_slot(og, s0);
                acc[s0] = acc[s1];
                jc[s0] = jc[s1];
#pragma unroll
                for (int b = 0; b < NB; ++b) acc[s1].v[b] = 0.0f;
            }
        o[AX][0] = o[AX][1];
        o[AX][1] = new_leading;
#pragma unroll
        for (int u = 0; u < 2; ++u)
#pragma unroll
            for (int v = 0; v < 2; ++v) {
                const int s1 = slot<AX>(1, u, v);
                jc[s1] = ld_bins<NB>(jg + off(s1));
            }
    }
};

template <int NB>
__global__ void __launch_bounds__(128) march_sliding_kernel(const MarchParams P) {
    RayId id;
    if (!ray_id(P, id)) return;
    RaySetup R = ray_setup(P, id);
    const int sx = P.ny * P.nz * P.nb, sy = P.nz * P.nb, sz = P.nb;
    const float* jg = P.j + id.group * NB;
    const float* kg = P.kappa + id.group * NB;
    float* og = P.out + id.group * NB;

    float I[NB], T[NB], att[NB];     // I scaled by 4 pi/N_Omega; T = exp(-tau); att = exp(-kappa ds) of the base cell
    Sliding<NB> S;
#pragma unroll
    for (int b = 0; b < NB; ++b) { I[b] = 0.0f; T[b] = 1.0f; att[b] = 1.0f; }
#pragma unroll
    for (int s = 0; s < 8; ++s)
#pragma unroll
        for (int b = 0; b < NB; ++b) S.acc[s].v[b] = 0.0f;
    // impossible offsets force a full (re)load at the first substep (nothing is flushed: acc is all zero)
    S.o[0][0] = S.o[0][1] = S.o[1][0] = S.o[1][1] = S.o[2][0] = S.o[2][1] = -1;

    for (int m = 0; m < P.n_steps; ++m) {
        for (int k = 0; k < P.n_sub; ++k) {
            const AxisTL ax = axis_tl(R.p[0], P.nx - 1, sx, R.neg[0]);
            const AxisTL ay = axis_tl(R.p[1], P.ny - 1, sy, R.neg[1]);
            const AxisTL az = axis_tl(R.p[2], P.nz - 1, sz, R.neg[2]);
            const bool cx = (ax.t != S.o[0][0]) | (ax.l != S.o[0][1]);
            const bool cy = (ay.t != S.o[1][0]) | (ay.l != S.o[1][1]);
            const bool cz = (az.t != S.o[2][0]) | (az.l != S.o[2][1]);
            if (cx | cy | cz) {
                // a slide by one cell keeps the old leading plane as the new trailing plane; anything else
                // (first substep, steps longer than a cell) restarts the stencil
                const bool jump = (cx & (ax.t != S.o[0][1])) | (cy & (ay.t != S.o[1][1])) |
                                  (cz & (az.t != S.o[2][1]));
                if (jump) {
                    S.flush_all(og);
                    S.o[0][0] = ax.t; S.o[0][1] = ax.l;
                    S.o[1][0] = ay.t; S.o[1][1] = ay.l;
                    S.o[2][0] = az.t; S.o[2][1] = az.l;
                    S.load_all(jg);
                } else {
                    if (cx) S.template shift<0>(og, jg, ax.l);
                    if (cy) S.template shift<1>(og, jg, ay.l);
                    if (cz) S.template shift<2>(og, jg, az.l);
                }
                // kappa: nearest neighbour at the base cell (lo, lo, lo) = the trailing index, or the leading
                // one on axes the ray descends (D4)
                const int base = S.o[0][R.neg[0] ? 1 : 0] + S.o[1][R.neg[1] ? 1 : 0] + S.o[2][R.neg[2] ? 1 : 0];
                const BinVec<NB> kap = ld_bins<NB>(kg + base);
#pragma unroll
                for (int b = 0; b < NB; ++b) att[b] = expf(-kap.v[b] * P.ds_f);
            }
            const float wx[2] = {ax.wt, ax.wl}, wy[2] = {ay.wt, ay.wl}, wz[2] = {az.wt, az.wl};
            float w[8];
            float jv[NB];
#pragma unroll
            for (int b = 0; b < NB; ++b) jv[b] = 0.0f;
#pragma unroll
            for (int s = 0; s < 8; ++s) {
                w[s] = wx[s >> 2] * wy[(s >> 1) & 1] * wz[s & 1];
#pragma unroll
                for (int b = 0; b < NB; ++b) jv[b] = fmaf(w[s], S.jc[s].v[b], jv[b]);
            }
#pragma unroll
            for (int b = 0; b < NB; ++b) {                       // eq. (2)
                I[b] = fmaf(I[b], att[b], jv[b] * T[b] * P.emis);
                T[b] *= att[b];
            }
#pragma unroll
            for (int s = 0; s < 8; ++s)
#pragma unroll
                for (int b = 0; b < NB; ++b) S.acc[s].v[b] = fmaf(w[s], I[b], S.acc[s].v[b]);
#pragma unroll
            for (int a = 0; a < 3; ++a) fx_add(R.p[a], R.d[a]);
        }
        S.flush_all(og);       // time-step boundary: snapshot m is complete (rays continue, D7)
        og += P.snap_stride;
    }
}

// ===================================================================================================
// set-up and post kernels
// ===================================================================================================
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

__global__ void directions_kernel(double* nhat, int n_rays) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_rays) return;
    double nh[3];
    fib_direction(uint32_t(i), uint32_t(n_rays), nh);
    nhat[3 * size_t(i)] = nh[0];
    nhat[3 * size_t(i) + 1] = nh[1];
    nhat[3 * size_t(i) + 2] = nh[2];
}

// out[m] <- out[0] + ... + out[m]: per-step increments become cumulative snapshots (D7)
__global__ void snapshot_prefix_kernel(float* out, long long stride, int n_steps) {
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < stride;
         e += (long long)gridDim.x * blockDim.x) {
        float run = out[e];
        for (int m = 1; m < n_steps; ++m) {
            run += out[m * stride + e];
            out[m * stride + e] = run;
        }
    }
}

}  // namespace rt
