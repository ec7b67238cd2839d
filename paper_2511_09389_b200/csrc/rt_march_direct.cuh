// rt_march_direct.cuh — the textbook form of the march (tests and bench only) and the single-ray trace hook.
// One thread marches one (source, direction, bin-group) ray in ARRAY coordinates: per substep 8 loads of j, 1 of
// kappa, eq. (2), and 8 reductions straight into the accumulation grid.
#pragma once
#include "rt_common.cuh"

namespace rt {

// per-axis clamped stencil (D5): lo = clamp(floor x), hi = clamp(floor x + 1),
// weights (1-f, f) from the unclamped fraction
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

struct RaySetup {
    Fx96 p[3], d[3];
};

__device__ __forceinline__ RaySetup ray_setup(const MarchParams& P, const RayId& id) {
    RaySetup r;
    double nh[3];
    fib_direction(id.index, uint32_t(P.n_rays), nh);
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        r.p[a] = fx_from_double(source_coord(P, id.src, a));
        r.d[a] = fx_from_double(__dmul_rn(P.ds, nh[a]));
    }
    return r;
}

template <int NB, typename ACC>
__global__ void __launch_bounds__(kThreads) march_direct_kernel(const MarchParams P) {
    RayId id;
    if (!ray_id(P, id)) return;
    RaySetup R = ray_setup(P, id);
    const int sx = P.ny * P.nz * P.nb, sy = P.nz * P.nb, sz = P.nb;
    const float* jg = P.j + id.group * NB;
    const float* kg = P.kappa + id.group * NB;
    ACC* og = static_cast<ACC*>(P.acc) + id.group * NB;
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
                red_bins(og + off[c], d);
            }
#pragma unroll
            for (int a = 0; a < 3; ++a) fx_add(R.p[a], R.d[a]);
        }
        og += P.snap_stride;
    }
}

// TEST HOOK: one thread marches one ray with the arithmetic above and records, per substep, the position x_k (as
// double: cell + 64-bit fraction), I_{k+1} (UNscaled by 4 pi/N_Omega) and T_{k+1} = exp(-tau_{k+1}) for every bin.
__global__ void trace_ray_kernel(const MarchParams P, uint32_t ray_index, int n_sub, double* pos, float* trI,
                                 float* trT) {
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

}  // namespace rt
