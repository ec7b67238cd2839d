// rt_march_sliding.cuh — the product march kernel (sm_100a): sliding-stencil register accumulation.
//
// One thread marches one (source, direction, bin-group) ray for all n_steps * N_s substeps of eq. (2)
// (PAPER.md:23).  The 8 voxels of the ray's clamped trilinear stencil live in registers: their j
// values (read once per voxel) and their pending deposits.  A voxel's pending deposit is reduced to memory
// (red.global.add) only when the stencil slides off it, so a ray issues ~1 reduction per substep instead of 8,
// and a ray that has left the box on all three axes issues one reduction for the rest of its path.  The sums are
// the same sums (each voxel still receives every w_c I_{k+1}); only their association changes.
//
// Each axis is handled in TRAVEL coordinates u = +x or u = -x (exact negation of the fixed-point position), so
// every axis ascends: the stencil's slots are (trailing, leading) per axis, a cell crossing is the carry out of
// the fraction, and a slide flushes the 4 trailing slots, moves 4, loads 4.  For a descending axis the array
// index of u-cell c is -c, the weight pair (trailing, leading) = (1 - frac u, frac u) is the oracle's
// (weight of hi, weight of lo), and floor(x) -- the nearest-neighbour kappa cell, PAPER.md:29 / D4 -- is the
// LEADING index unless frac u = 0 exactly, when it is the trailing one (and the leading slot has weight 0 where
// the array-coordinate stencil has its weight-0 hi corner: the same field).
//
// Clamping (D5): where both indices of an axis clamp to the same voxel the two slots are merged
// (weights (1, 0)); nothing slides while the ray moves on outside the box.
#pragma once
#include "rt_common.cuh"

namespace rt {

// accumulator / j-cache slot for (plane p of axis AX, other two axes u, v); slots are [x][y][z], 0 = trailing
template <int AX> __device__ __forceinline__ constexpr int slot(int p, int u, int v) {
    return AX == 0 ? (p * 4 + u * 2 + v) : (AX == 1 ? (u * 4 + p * 2 + v) : (u * 4 + v * 2 + p));
}

struct TravelAxis {
    Fx96 p, d;          // position and per-substep increment in travel coordinates (d >= 0)
    int t, dl;          // element offset of the trailing index; leading minus trailing offset (0 = merged)
    int stride, nmax;   // element stride of this axis, N - 1
    bool neg;           // the ray descends this axis (u = -x)

    __device__ __forceinline__ int eoff(int c) const {          // element offset of u-cell c, index clamped
        const int idx = neg ? -c : c;
        return min(max(idx, 0), nmax) * stride;
    }
    __device__ __forceinline__ bool on_a_plane() const { return (p.fh | p.fl) == 0u; }
};

template <int NB, typename ACC> struct Stencil {
    BinVec<NB> acc[8];   // pending deposits for the 8 stencil voxels
    BinVec<NB> jc[8];    // j at the 8 stencil voxels
    int off[8];          // their element offsets

    __device__ __forceinline__ void flush_slot(ACC* og, int s) {
        if (any_nonzero<NB>(acc[s])) red_bins(og + off[s], acc[s]);
    }
    __device__ __forceinline__ void zero_slot(int s) {
#pragma unroll
        for (int b = 0; b < NB; ++b) acc[s].v[b] = 0.0f;
    }
    __device__ __forceinline__ void flush_all(ACC* og) {
#pragma unroll
        for (int s = 0; s < 8; ++s) {
            flush_slot(og, s);
            zero_slot(s);
        }
    }
    // (re)build the stencil at the axes' current cells; pending deposits must have been flushed
    __device__ __forceinline__ void restart(TravelAxis (&A)[3], const float* jg) {
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            A[a].t = A[a].eoff(A[a].p.c);
            A[a].dl = A[a].eoff(A[a].p.c + 1) - A[a].t;
        }
#pragma unroll
        for (int s = 0; s < 8; ++s) {
            off[s] = A[0].t + A[1].t + A[2].t + ((s & 4) ? A[0].dl : 0) + ((s & 2) ? A[1].dl : 0) +
                     ((s & 1) ? A[2].dl : 0);
            jc[s] = ld_bins<NB>(jg + off[s]);
        }
    }
    // axis AX advanced by one cell.  move: the trailing index changed (the old leading plane is the new trailing
    // plane); load: the leading plane holds new voxels; dl: new leading-minus-trailing offset
    template <int AX> __device__ __forceinline__ void slide(ACC* og, const float* jg, bool move, bool load, int dl) {
#pragma unroll
        for (int u = 0; u < 2; ++u)
#pragma unroll
            for (int v = 0; v < 2; ++v) {
                const int s0 = slot<AX>(0, u, v), s1 = slot<AX>(1, u, v);
                if (move) {
                    flush_slot(og, s0);
                    acc[s0] = acc[s1];
                    jc[s0] = jc[s1];
                    off[s0] = off[s1];
                    zero_slot(s1);
                }
                off[s1] = off[s0] + dl;
                if (load) jc[s1] = ld_bins<NB>(jg + off[s1]);
            }
    }
    template <int AX> __device__ __forceinline__ void axis_step(TravelAxis& A, ACC* og, const float* jg) {
        const int tn = A.eoff(A.p.c), dln = A.eoff(A.p.c + 1) - tn;
        const bool move = (tn != A.t);
        const bool load = (dln != 0) & (move | (dln != A.dl));
        if (move | load) slide<AX>(og, jg, move, load, dln);
        A.t = tn;
        A.dl = dln;
    }
};

template <int NB, typename ACC>
__global__ void __launch_bounds__(kThreads) march_sliding_kernel(const MarchParams P) {
    RayId id;
    if (!ray_id(P, id)) return;
    const float* jg = P.j + id.group * NB;
    const float* kg = P.kappa + id.group * NB;
    ACC* og = static_cast<ACC*>(P.acc) + id.group * NB;

    TravelAxis A[3];
    {
        double nh[3];
        fib_direction(id.index, uint32_t(P.n_rays), nh);
        const int strides[3] = {P.ny * P.nz * P.nb, P.nz * P.nb, P.nb}, nmaxs[3] = {P.nx - 1, P.ny - 1, P.nz - 1};
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            A[a].neg = nh[a] < 0.0;
            A[a].p = fx_from_double(source_coord(P, id.src, a), A[a].neg);
            A[a].d = fx_from_double(__dmul_rn(P.ds, nh[a]), A[a].neg);
            A[a].stride = strides[a];
            A[a].nmax = nmaxs[a];
        }
    }
    Stencil<NB, ACC> S;
#pragma unroll
    for (int s = 0; s < 8; ++s) S.zero_slot(s);
    S.restart(A, jg);

    float I[NB], T[NB], att[NB];     // I scaled by 4 pi/N_Omega; T = exp(-tau); att = exp(-kappa ds) of the kappa cell
#pragma unroll
    for (int b = 0; b < NB; ++b) { I[b] = 0.0f; T[b] = 1.0f; att[b] = 1.0f; }
    int kof = -1;                    // element offset of the kappa cell att[] belongs to
    bool refresh = true;             // re-derive the kappa cell before the next substep

    for (int m = 0; m < P.n_steps; ++m) {
        for (int k = 0; k < P.n_sub; ++k) {
            if (refresh) {
                // kappa: nearest neighbour at clamp(floor(x_k)) (D4): the trailing index, or the
                // leading one on an axis the ray descends unless it sits exactly on a cell plane -- then the
                // cell changes at the next substep with no slide, so look again
                int ko = S.off[0];
                refresh = false;
#pragma unroll
                for (int a = 0; a < 3; ++a)
                    if (A[a].neg) {
                        if (A[a].on_a_plane()) refresh = true;
                        else ko += A[a].dl;
                    }
                if (ko != kof) {
                    kof = ko;
                    const BinVec<NB> kap = ld_bins<NB>(kg + ko);
#pragma unroll
                    for (int b = 0; b < NB; ++b) att[b] = expf(-kap.v[b] * P.ds_f);
                }
            }
            // trilinear weights from the top 32 fraction bits: leading f, trailing 1 - f (each truncated to the
            // 2^-32 grid, so tiny weights keep their relative accuracy); merged axes carry (1, 0)
            float wt[3], wl[3];
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const float f = __uint2float_rn(A[a].p.fh) * 2.3283064365386963e-10f;      // 2^-32
                const float g = __uint2float_rn(~A[a].p.fh) * 2.3283064365386963e-10f;
                const bool merged = (A[a].dl == 0);
                wl[a] = merged ? 0.0f : f;
                wt[a] = merged ? 1.0f : g;
            }
            const float wxy[4] = {wt[0] * wt[1], wt[0] * wl[1], wl[0] * wt[1], wl[0] * wl[1]};
            float w[8];
            float jv[NB];
#pragma unroll
            for (int b = 0; b < NB; ++b) jv[b] = 0.0f;
#pragma unroll
            for (int s = 0; s < 8; ++s) {
                w[s] = wxy[s >> 1] * ((s & 1) ? wl[2] : wt[2]);
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

            // x_{k+1} = x_k + n ds; a changed cell word is a crossing (increments are >= 0 in travel coordinates)
            const int c0 = A[0].p.c, c1 = A[1].p.c, c2 = A[2].p.c;
#pragma unroll
            for (int a = 0; a < 3; ++a) fx_add(A[a].p, A[a].d);
            const int d0 = A[0].p.c - c0, d1 = A[1].p.c - c1, d2 = A[2].p.c - c2;
            if (d0 | d1 | d2) {
                if ((d0 | d1 | d2) > 1) {          // a step longer than a cell: restart the stencil
                    S.flush_all(og);
                    S.restart(A, jg);
                } else {
                    if (d0) S.template axis_step<0>(A[0], og, jg);
                    if (d1) S.template axis_step<1>(A[1], og, jg);
                    if (d2) S.template axis_step<2>(A[2], og, jg);
                }
                refresh = true;
            }
        }
        S.flush_all(og);       // time-step boundary: the increments of step m are complete (rays continue, D7)
        og += P.snap_stride;
    }
}

}  // namespace rt
