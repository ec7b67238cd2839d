// rt_adjoint.cuh — adjoints of the march with respect to j and to kappa (reading D19),
// sm_100a.  The j part first; the kappa part is described at adjoint_kernel.
//
// For fixed kappa the field is linear in j.  With gbar[m] = dL/d out[m] and gsuf[m] = sum_{m' >= m} gbar[m'] (the
// snapshots are cumulative, D7), eq. (2) and the deposit rule give, per ray,
//     lambda_{k+1} = s (w_k . gsuf[step(k)]) + a_{k+1} lambda_{k+2},   lambda_{K+1} = 0,   s = 4 pi / N_Omega
//     grad_j[corner_c] += lambda_{k+1} T_k ds w_k[c],                  a_k = exp(-kappa_k ds), T_k = exp(-tau_k)
// i.e. the SAME sliding-stencil march run backwards along the ray: the gather reads gsuf instead of j, the carried
// scalar is lambda instead of I, and what is deposited (same weights, same clamped corners) is lambda T_k ds.
//
// One thread = one (source, direction, bin).  Phase 1 walks the ray forwards reading only kappa and sums tau_K in
// fp64.  Phase 2 walks it backwards from x_{K-1}: a ray with direction -n, so an axis the forward ray ascends is
// marched in the complement travel coordinate and vice versa (rt_march_sliding.cuh); the fixed-point positions are
// the forward ray's, bit for bit, hence the same cells and the same weight bits.  tau_k is recovered by
// subtracting kappa_k ds in fp64 (an fp32 running difference would lose 1e-3 of T over a few hundred substeps).
#pragma once
#include "rt_march_phased.cuh"
#include "rt_march_sliding.cuh"

namespace rt {

// WRT_KAPPA = false: dL/dj as described above.  WRT_KAPPA = true: dL/dkappa (D19).  Unrolling eq. (2),
// I_{k+1} = T_{k+1} sum_{m<=k} ds J_m / a_m, so with G_k = w_k . gsuf and P_i = ds J_i T_i (the emission term of
// substep i) dL/dkappa_i = ds [P_i lambda_{i+1} - R_i], R_i = sum_{k>=i} G_k I_{k+1}: the same backward march,
// fed with I_{k+1} of every substep as recorded by march_phased_kernel<..., RECORD = true> (P_k = I_{k+1} - a_k I_k), summing into the kappa cell of x_i
// (nearest neighbour: one voxel per substep, reduced when the cell changes).
#ifndef RT_REC_AHEAD
#define RT_REC_AHEAD 8
#endif
// The kappa adjoint reads the forward record of substep kk - 1 into a register while it works on substep kk, and asks
// the L2 for the record of substep kk - kRecAhead (a register queue deeper than one does not help: moving a value
// along the queue waits for its load)
constexpr int kRecAhead = RT_REC_AHEAD;

// The state one lane carries through the backward march
struct AdjointLane {
    Stencil<1, double, false> S;     // cached gsuf values (jc) and pending deposits (acc)
    TravelAxis A[3];
    float lambda, a_next, kap;       // kap: kappa of the cell of x_k as loaded; exp(-kappa ds) is formed where it is used, a
                                     // substep after the load
    double tau, Rsum, kacc;          // WRT_KAPPA: R_i and the pending sum of the current kappa cell, in fp64 (P_i lambda_{i+1} - R_i cancels)
    int ko;                          // element offset of the kappa cell
    long long kk;                    // global substep index of the backward sweep
    float rec, rec1;                 // WRT_KAPPA: the records I_{kk+1} and I_kk, loaded one and two substeps before this one
    int left;                        // substeps left in the current time step
    float* sg;                       // BRICK: the fp32 window-brick scratch (rt_brick.cuh) the dL/dj deposits go to ...
    int woff;                        // ... and the float offset in it of the window the trailing slots start
};

// PHASES of the backward march (cf. rt_march_phased.cuh).  The backward ray starts at x_{K-1}, for most rays far outside
// the box, and comes in: an axis is INACTIVE for a warp while every lane is still short of the face it will enter
// through (travel cell word below the near face, by a margin of kAdjMargin cells: the test runs every 4th substep and a
// substep is shorter than a cell) -- merged, weights exactly (1, 0), leading slots never touched and exactly zero.
// adjoint_phase<ACT> is the substep loop with those axes compiled out; it returns the new set of active axes (one more
// axis: a warp vote), or ACT at a time-step boundary.  Activation needs no reload: no lane has entered yet, so the
// axis is still merged in every lane and its first slide loads its leading slots.
constexpr int kAdjMargin = 4;

template <int ACT, bool WRT_KAPPA, bool BRICK>
__device__ __forceinline__ int adjoint_phase(const MarchParams& P, const BrickGeom& G, AdjointLane& L, int negbits, double* og, const float* gs,
                                             const float* fwd, long long fwd_stride, long long tid, int bin, bool live) {
    constexpr int kBits = ((ACT & 1) ? 4 : 0) | ((ACT & 2) ? 2 : 0) | ((ACT & 4) ? 1 : 0);
    constexpr int kActive = ((ACT & 1) ? 1 : 0) + ((ACT & 2) ? 1 : 0) + ((ACT & 4) ? 1 : 0);
    constexpr int kLast = (ACT & 4) ? 2 : ((ACT & 2) ? 1 : 0);
    auto load_kappa = [&]() {
        int ko = L.S.base;
        if (ACT & 1) ko += (negbits & 1) ? L.A[0].dl : 0;
        if (ACT & 2) ko += (negbits & 2) ? L.A[1].dl : 0;
        if (ACT & 4) ko += (negbits & 4) ? L.A[2].dl : 0;
        L.ko = ko;
        L.kap = __ldg(P.kappa + ko);
    };
    int next = ACT;
    do {
        float w[8];
        bool cross[3] = {false, false, false};
        {
            float t[3] = {1.0f, 1.0f, 1.0f}, l[3] = {0.0f, 0.0f, 0.0f};
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                if (ACT & (1 << a)) {
                    const uint32_t h = L.A[a].p.fh & L.A[a].fmask;
                    const float sc = (a == kLast) ? (kActive == 3 ? 1.2621774483536189e-29f
                                                                  : (kActive == 2 ? 5.421010862427522e-20f : 2.3283064365386963e-10f))
                                                  : 1.0f;
                    t[a] = __uint2float_rn(~h) * sc;
                    l[a] = __uint2float_rn(h) * sc;
                }
                const int c = L.A[a].p.c;                  // every axis is advanced: an inactive one is watched for its entry
                fx_add(L.A[a].p, L.A[a].d);
                cross[a] = (ACT & (1 << a)) && L.A[a].p.c != c;
            }
            const float wx[2] = {t[0], l[0]}, wy[2] = {t[1], l[1]}, wz[2] = {t[2], l[2]};
#pragma unroll
            for (int s = 0; s < 8; ++s)
                if ((s & ~kBits) == 0) {
                    float v = 1.0f;
                    bool first = true;
                    if (ACT & 1) { v = wx[s >> 2]; first = false; }
                    if (ACT & 2) { v = first ? wy[(s >> 1) & 1] : v * wy[(s >> 1) & 1]; first = false; }
                    if (ACT & 4) { v = first ? wz[s & 1] : v * wz[s & 1]; }
                    w[s] = v;
                }
        }
        float gv = 0.0f, gu = 0.0f;
#pragma unroll
        for (int s = 0; s < 8; ++s)
            if ((s & ~kBits) == 0) {
                const int r = slot_rank(s, kBits);
                const float g = L.S.jc[s].v[0];
                if (r & 1) gu = (r == 1) ? w[s] * g : fmaf(w[s], g, gu);
                else gv = (r == 0) ? w[s] * g : fmaf(w[s], g, gv);
            }
        if (!live) { gv = 0.0f; gu = 0.0f; }         // a dark lane: zero dL/d out, so lambda stays 0 and nothing is deposited
        if (WRT_KAPPA) {
            // The record holds I_{k+1} (x 4 pi/N_Omega) of every substep; the emission term is recovered from two of them,
            // P_k = I_{k+1} - a_k I_k (eq. (2) solved for it; off by the rounding of the forward fma, <= 2^-25 I_{k+1}).
            // I_{k+1} and I_k were loaded one and two substeps ago; the load issued now is I_{k-1}.  (A dark lane: zeros.)
            const float I_next = L.rec, I_cur = L.rec1;
            L.rec = I_cur;
            L.rec1 = (live && L.kk >= 2) ? __ldg(fwd + (L.kk - 2) * fwd_stride + tid) : 0.0f;
            if (live && L.kk >= kRecAhead) asm volatile("prefetch.global.L2 [%0];" ::"l"(fwd + (L.kk - kRecAhead) * fwd_stride + tid));
            L.lambda = fmaf(L.a_next, L.lambda, gv + gu);
            L.a_next = ex2_approx(L.kap * P.att_scale);                          // a_k, the same bits as in the forward march
            const float P_k = fmaf(-L.a_next, I_cur, I_next);
            L.Rsum = fma(double(gv + gu), double(I_next), L.Rsum);
            L.kacc = fma(fma(double(P_k), double(L.lambda), -L.Rsum), P.ds, L.kacc);
            --L.kk;
        } else {
            L.tau = fma(-double(L.kap), P.ds, L.tau);                             // tau_k = tau_{k+1} - kappa_k ds
            const float T = ex2_approx(float(L.tau * -1.4426950408889634));       // exp(-tau_k)
            L.lambda = fmaf(L.a_next, L.lambda, (gv + gu) * P.emis);              // lambda_{k+1} ds
            L.a_next = ex2_approx(L.kap * P.att_scale);
            const float v = L.lambda * T;
#pragma unroll
            for (int s = 0; s < 8; ++s)
                if ((s & ~kBits) == 0) L.S.acc[s].v[0] = (ACT == 0) ? L.S.acc[s].v[0] + v : fmaf(w[s], v, L.S.acc[s].v[0]);
        }
        if (cross[0] | cross[1] | cross[2]) {
            bool jumped = false;
            if constexpr (ACT == 7) {            // a substep of a cell or more (all axes active then) may cross two planes
                if (P.ds_f >= 1.0f) {
                    const int c0 = L.A[0].p.c, c1 = L.A[1].p.c, c2 = L.A[2].p.c;
                    // cell words one substep ago: position minus increment (travel increments are >= 0)
                    Fx96 q0 = L.A[0].p, q1 = L.A[1].p, q2 = L.A[2].p;
                    fx_sub(q0, L.A[0].d); fx_sub(q1, L.A[1].d); fx_sub(q2, L.A[2].d);
                    jumped = ((c0 - q0.c) | (c1 - q1.c) | (c2 - q2.c)) > 1;
                    if (jumped) {
                        L.S.flush_all(og, L.A);
                        L.S.restart(P, L.A, negbits, bin, gs);
                    }
                }
            }
            if (!jumped) {               // slides with the loads deferred (rt_march_sliding.cuh)
                uint32_t stale = 0;
                // the trailing plane goes slot by slot into the fp64 grid, or as one vector reduction into the brick scratch
                if (cross[0]) L.S.template axis_slide_deferred<0, ACT>(P, L.A, negbits, stale, [&]() {
                    if constexpr (BRICK) brick_flush<0, ACT>(G, L, negbits); else L.S.template flush_trailing<0, ACT>(og, L.A); });
                if (cross[1]) L.S.template axis_slide_deferred<1, ACT>(P, L.A, negbits, stale, [&]() {
                    if constexpr (BRICK) brick_flush<1, ACT>(G, L, negbits); else L.S.template flush_trailing<1, ACT>(og, L.A); });
                if (cross[2]) L.S.template axis_slide_deferred<2, ACT>(P, L.A, negbits, stale, [&]() {
                    if constexpr (BRICK) brick_flush<2, ACT>(G, L, negbits); else L.S.template flush_trailing<2, ACT>(og, L.A); });
                L.S.template load_stale<ACT>(P, L.A, gs, stale);
            }
            if (WRT_KAPPA) {                     // the kappa cell may have changed: reduce the old one's sum
                const int ko_old = L.ko;
                load_kappa();
                if (L.ko != ko_old) {
                    if (L.kacc != 0.0)
                        asm volatile("red.global.add.f64 [%0], %1;" ::"l"(og + ko_old), "d"(L.kacc) : "memory");
                    L.kacc = 0.0;
                }
            } else {
                load_kappa();
            }
        }
        --L.left;
        if constexpr (ACT != 7) {
            if ((L.left & 3) == 0) {             // is a lane about to enter through an inactive axis?
#pragma unroll
                for (int a = 0; a < 3; ++a)
                    if (!(ACT & (1 << a))) {
                        const int lim = (a == 0 ? P.nx : (a == 1 ? P.ny : P.nz)) - 1;
                        const bool near = L.A[a].p.c + kAdjMargin >= ((negbits & (1 << a)) ? -lim : 0);
                        if (__any_sync(0xFFFFFFFFu, near)) next |= 1 << a;
                    }
            }
        }
    } while (L.left != 0 && next == ACT);
    return next;
}

// WRT_KAPPA = false: dL/dj as described above.  WRT_KAPPA = true: dL/dkappa (D19).  Unrolling eq. (2),
// I_{k+1} = T_{k+1} sum_{m<=k} ds J_m / a_m, so with G_k = w_k . gsuf and P_i = ds J_i T_i (the emission term of
// substep i) dL/dkappa_i = ds [P_i lambda_{i+1} - R_i], R_i = sum_{k>=i} G_k I_{k+1}: the same backward march,
// fed with I_{k+1} of every substep as recorded by march_phased_kernel<..., RECORD = true> (P_k = I_{k+1} - a_k I_k), summing into the kappa cell of x_i
// (nearest neighbour: one voxel per substep, reduced when the cell changes).
// this block's turn at the drain of the brick scratch (as at the end of march_phased_kernel)
__device__ __forceinline__ void adjoint_drain_slice(const MarchParams& P, const BrickGeom& G) {
    const long long per = P.drain_units_per_block;
    if (per == 0) return;
    const long long n_slices = (P.n_drain_units + per - 1) / per;
    const long long b0 = (blockIdx.x % n_slices) * per;
    drain_bricks(P.scratch, static_cast<double*>(P.acc), G, P.nx, P.ny, P.nz, b0, min(b0 + per, P.n_drain_units), threadIdx.x, kThreads);
}

// BRICK (dL/dj, one bin, substeps shorter than a cell): the deposits go to the fp32 window-brick scratch P.scratch with one
// vector reduction per stencil plane and every block drains a slice of it into the fp64 grid when its rays are done, as
// in the forward march (rt_brick.cuh, rt_march_phased.cuh).
// ONE_DIR: every warp marches one direction (map_src = 1): the direction signs pass through a vote and live in uniform
// registers, as in march_phased_kernel (dL/dj 16.8 -> 16.5 ms, dL/dkappa 27.3 -> 26.9 on C2).
template <int MINB, bool WRT_KAPPA, bool BRICK = false, bool ONE_DIR = false>
__global__ void __launch_bounds__(kThreads, MINB) adjoint_kernel(const MarchParams P, const float* gsuf,
                                                                 const float* fwd, long long fwd_stride) {
    // a warp marches as a whole (its phases are warp votes): a lane without a ray of its own marches the ray of the
    // warp's first live lane with gsuf read as zero weight -- lambda stays 0, nothing is deposited
    RayId id;
    const bool live = ray_id(P, id);
    const unsigned live_mask = __ballot_sync(0xFFFFFFFFu, live);
    const BrickGeom G = brick_geom(P.nx, P.ny, P.nz);
    if (!live_mask) {
        if constexpr (BRICK) adjoint_drain_slice(P, G);
        return;
    }
    {
        const int leader = __ffs(live_mask) - 1;
        const int lsrc = __shfl_sync(0xFFFFFFFFu, id.src, leader), lgroup = __shfl_sync(0xFFFFFFFFu, id.group, leader);
        const uint32_t lindex = __shfl_sync(0xFFFFFFFFu, id.index, leader);
        if (!live) { id.src = lsrc; id.group = lgroup; id.index = lindex; }
    }
    const long long tid = (long long)blockIdx.x * kThreads + threadIdx.x;
    const int bin = id.group;                       // one bin per thread (n_groups = n_bins)
    double* og = static_cast<double*>(P.acc);

    Fx96 X[3], D[3];
    bool fwd_neg[3];
    {
        double nh[3];
        fib_direction(id.index, uint32_t(P.n_rays), nh);
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            fwd_neg[a] = nh[a] < 0.0;
            X[a] = fx_from_double(source_coord(P, id.src, a));
            D[a] = fx_from_double(__dmul_rn(P.ds, nh[a]));
        }
    }
    // phase 1: tau_K = ds * sum_k kappa(cell of x_k), forwards (nearest neighbour, clamped: PAPER.md:29, D4)
    const int sx = P.ny * P.nz * P.nb, sy = P.nz * P.nb, sz = P.nb;
    AdjointLane L;
    L.tau = 0.0;
    const long long K = (long long)P.n_steps * P.n_sub;
    if (WRT_KAPPA) {                                 // tau is not needed: jump to x_K
#pragma unroll
        for (int a = 0; a < 3; ++a) fx_advance(X[a], D[a], K);
    } else {
        for (long long k = 0; k < K; ++k) {
            const int o = min(max(X[0].c, 0), P.nx - 1) * sx + min(max(X[1].c, 0), P.ny - 1) * sy +
                          min(max(X[2].c, 0), P.nz - 1) * sz;
            L.tau = fma(double(__ldg(P.kappa + o + bin)), P.ds, L.tau);
#pragma unroll
            for (int a = 0; a < 3; ++a) fx_add(X[a], D[a]);
        }
    }
    // phase 2: backwards from x_{K-1}
    int negbits = 0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        Fx96 nd;                                     // -D, exact
        nd.fl = 0u - D[a].fl;
        nd.fh = ~D[a].fh + (nd.fl == 0u ? 1u : 0u);
        nd.c = ~D[a].c + ((nd.fl == 0u && nd.fh == 0u) ? 1 : 0);
        fx_add(X[a], nd);                            // x_{K-1}
        if (fwd_neg[a]) {                            // the backward ray ascends this axis
            L.A[a].p = X[a];
            L.A[a].d = nd;
        } else {                                     // it descends: complement coordinate, increment +D
            L.A[a].p.c = ~X[a].c; L.A[a].p.fh = ~X[a].fh; L.A[a].p.fl = ~X[a].fl;
            L.A[a].d = D[a];
            negbits |= 1 << a;
        }
    }
    asm volatile("" : "+r"(negbits));
    if constexpr (ONE_DIR)
        negbits = (__any_sync(0xFFFFFFFFu, (negbits & 1) != 0) ? 1 : 0) | (__any_sync(0xFFFFFFFFu, (negbits & 2) != 0) ? 2 : 0) |
                  (__any_sync(0xFFFFFFFFu, (negbits & 4) != 0) ? 4 : 0);
#pragma unroll
    for (int s = 0; s < 8; ++s) L.S.zero_slot(s);
    const float* gs = gsuf + (long long)(P.n_steps - 1) * P.snap_stride;
    L.S.restart(P, L.A, negbits, bin, gs);
    L.sg = P.scratch;
    L.woff = 0;
    if constexpr (BRICK)
        L.woff = (aidx<0>(P, L.A[0].p.c, negbits) * G.wy + aidx<1>(P, L.A[1].p.c, negbits) + ((negbits & 2) ? 0 : 1)) * G.sy +
                 (aidx<2>(P, L.A[2].p.c, negbits) + ((negbits & 4) ? 0 : 1)) * 4;
    L.lambda = 0.0f; L.a_next = 0.0f;
    L.Rsum = 0.0; L.kacc = 0.0;
    L.ko = L.S.base + ((negbits & 1) ? L.A[0].dl : 0) + ((negbits & 2) ? L.A[1].dl : 0) + ((negbits & 4) ? L.A[2].dl : 0);
    L.kap = __ldg(P.kappa + L.ko);
    L.kk = K - 1;
    L.rec = (WRT_KAPPA && live) ? __ldg(fwd + (K - 1) * fwd_stride + tid) : 0.0f;
    L.rec1 = (WRT_KAPPA && live && K >= 2) ? __ldg(fwd + (K - 2) * fwd_stride + tid) : 0.0f;
    L.left = P.n_sub;
    // axes some lane is inside of, or about to enter, at x_{K-1}
    int act = 0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const int lim = (a == 0 ? P.nx : (a == 1 ? P.ny : P.nz)) - 1;
        const bool near = L.A[a].p.c + kAdjMargin >= ((negbits & (1 << a)) ? -lim : 0);
        if (__any_sync(0xFFFFFFFFu, near)) act |= 1 << a;
    }
    if (!(P.ds_f < 1.0f)) act = 7;                   // substeps of a cell or more: no phases (the margin assumes shorter ones)
    int m = P.n_steps - 1;
    while (true) {
        {
            switch (act) {
                case 7: act = adjoint_phase<7, WRT_KAPPA, BRICK>(P, G, L, negbits, og, gs, fwd, fwd_stride, tid, bin, live); break;
                case 6: act = adjoint_phase<6, WRT_KAPPA, BRICK>(P, G, L, negbits, og, gs, fwd, fwd_stride, tid, bin, live); break;
                case 5: act = adjoint_phase<5, WRT_KAPPA, BRICK>(P, G, L, negbits, og, gs, fwd, fwd_stride, tid, bin, live); break;
                case 4: act = adjoint_phase<4, WRT_KAPPA, BRICK>(P, G, L, negbits, og, gs, fwd, fwd_stride, tid, bin, live); break;
                case 3: act = adjoint_phase<3, WRT_KAPPA, BRICK>(P, G, L, negbits, og, gs, fwd, fwd_stride, tid, bin, live); break;
                case 2: act = adjoint_phase<2, WRT_KAPPA, BRICK>(P, G, L, negbits, og, gs, fwd, fwd_stride, tid, bin, live); break;
                case 1: act = adjoint_phase<1, WRT_KAPPA, BRICK>(P, G, L, negbits, og, gs, fwd, fwd_stride, tid, bin, live); break;
                default: act = adjoint_phase<0, WRT_KAPPA, BRICK>(P, G, L, negbits, og, gs, fwd, fwd_stride, tid, bin, live); break;
            }
        }
        if (L.left == 0) {                           // an earlier time step sees the suffix sum of one more snapshot
            if (--m < 0) break;
            gs -= P.snap_stride;
            L.S.reload(P, L.A, gs);
            L.left = P.n_sub;
        }
    }
    if (WRT_KAPPA) {
        if (L.kacc != 0.0) asm volatile("red.global.add.f64 [%0], %1;" ::"l"(og + L.ko), "d"(L.kacc) : "memory");
    } else if constexpr (BRICK) {
        brick_flush<-1, 7>(G, L, negbits);
        adjoint_drain_slice(P, G);
    } else {
        L.S.flush_all(og, L.A);
    }
}

// gsuf[m] = gbar[m] + gbar[m+1] + ... (the snapshots of the forward march are cumulative, D7)
__global__ void suffix_sum_kernel(const float* gbar, float* gsuf, long long stride, int n_steps) {
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < stride;
         e += (long long)gridDim.x * blockDim.x) {
        float run = 0.0f;
        for (int m = n_steps - 1; m >= 0; --m) {
            run += gbar[m * stride + e];
            gsuf[m * stride + e] = run;
        }
    }
}

}  // namespace rt
