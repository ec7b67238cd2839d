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
#include "rt_march_sliding.cuh"

namespace rt {

// WRT_KAPPA = false: dL/dj as described above.  WRT_KAPPA = true: dL/dkappa (D19).  Unrolling eq. (2),
// I_{k+1} = T_{k+1} sum_{m<=k} ds J_m / a_m, so with G_k = w_k . gsuf and P_i = ds J_i T_i (the emission term of
// substep i) dL/dkappa_i = ds [P_i lambda_{i+1} - R_i], R_i = sum_{k>=i} G_k I_{k+1}: the same backward march,
// fed with (I_{k+1}, P_k) of every substep as recorded by march_sliding_kernel<..., RECORD = true>, summing into the kappa cell of x_i
// (nearest neighbour: one voxel per substep, reduced when the cell changes).
template <int MINB, bool WRT_KAPPA>
__global__ void __launch_bounds__(kThreads, MINB) adjoint_kernel(const MarchParams P, const float* gsuf,
                                                                 const float2* fwd, long long fwd_stride) {
    RayId id;
    if (!ray_id(P, id)) return;
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
    double tau = 0.0;
    const long long K = (long long)P.n_steps * P.n_sub;
    if (WRT_KAPPA) {                                 // tau is not needed: jump to x_K
#pragma unroll
        for (int a = 0; a < 3; ++a) fx_advance(X[a], D[a], K);
    } else {
        for (long long k = 0; k < K; ++k) {
            const int o = min(max(X[0].c, 0), P.nx - 1) * sx + min(max(X[1].c, 0), P.ny - 1) * sy +
                          min(max(X[2].c, 0), P.nz - 1) * sz;
            tau = fma(double(__ldg(P.kappa + o + bin)), P.ds, tau);
#pragma unroll
            for (int a = 0; a < 3; ++a) fx_add(X[a], D[a]);
        }
    }
    // phase 2: backwards from x_{K-1}
    TravelAxis A[3];
    int negbits = 0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        Fx96 nd;                                     // -D, exact
        nd.fl = 0u - D[a].fl;
        nd.fh = ~D[a].fh + (nd.fl == 0u ? 1u : 0u);
        nd.c = ~D[a].c + ((nd.fl == 0u && nd.fh == 0u) ? 1 : 0);
        fx_add(X[a], nd);                            // x_{K-1}
        if (fwd_neg[a]) {                            // the backward ray ascends this axis
            A[a].p = X[a];
            A[a].d = nd;
        } else {                                     // it descends: complement coordinate, increment +D
            A[a].p.c = ~X[a].c; A[a].p.fh = ~X[a].fh; A[a].p.fl = ~X[a].fl;
            A[a].d = D[a];
            negbits |= 1 << a;
        }
    }
    asm volatile("" : "+r"(negbits));
    Stencil<1, double, false> S;
#pragma unroll
    for (int s = 0; s < 8; ++s) S.zero_slot(s);
    const float* gs = gsuf + (long long)(P.n_steps - 1) * P.snap_stride;
    S.restart(P, A, negbits, bin, gs);

    float lambda = 0.0f, a_next = 0.0f, kap = 0.0f, att = 1.0f;
    double Rsum = 0.0, kacc = 0.0;                   // WRT_KAPPA: R_i and the pending sum for the current kappa cell (fp64:
                                                     // P_i lambda_{i+1} - R_i cancels)
    int ko = 0;
    auto load_kappa = [&]() {
        ko = S.base + ((negbits & 1) ? A[0].dl : 0) + ((negbits & 2) ? A[1].dl : 0) + ((negbits & 4) ? A[2].dl : 0);
        kap = __ldg(P.kappa + ko);
        att = ex2_approx(kap * P.att_scale);
    };
    auto flush_kappa = [&]() {
        if (kacc != 0.0) asm volatile("red.global.add.f64 [%0], %1;" ::"l"(og + ko), "d"(kacc) : "memory");
        kacc = 0.0;
    };
    load_kappa();
    long long kk = K - 1;                            // global substep index of the backward sweep

    for (int m = P.n_steps - 1; m >= 0; --m) {
        if (m != P.n_steps - 1) {                    // an earlier time step sees the suffix sum of one more snapshot
            gs -= P.snap_stride;
            S.reload(P, A, gs);
        }
        for (int k = P.n_sub - 1; k >= 0; --k) {
            const uint32_t hx = A[0].p.fh & A[0].fmask, hy = A[1].p.fh & A[1].fmask, hz = A[2].p.fh & A[2].fmask;
            const float lx = __uint2float_rn(hx), tx = __uint2float_rn(~hx);
            const float ly = __uint2float_rn(hy), ty = __uint2float_rn(~hy);
            const float wz[2] = {__uint2float_rn(~hz) * 1.2621774483536189e-29f,      // 2^-96
                                 __uint2float_rn(hz) * 1.2621774483536189e-29f};
            const float wxy[4] = {tx * ty, tx * ly, lx * ty, lx * ly};
            float w[8];
#pragma unroll
            for (int s = 0; s < 8; ++s) w[s] = wxy[s >> 1] * wz[s & 1];
            float gv = w[0] * S.jc[0].v[0], gu = w[1] * S.jc[1].v[0];
#pragma unroll
            for (int s = 2; s < 8; s += 2) {
                gv = fmaf(w[s], S.jc[s].v[0], gv);
                gu = fmaf(w[s + 1], S.jc[s + 1].v[0], gu);
            }
            if (WRT_KAPPA) {
                const float2 rec = __ldg(fwd + kk * fwd_stride + tid);            // (I_{k+1}, P_k), both x 4 pi/N_Omega
                lambda = fmaf(a_next, lambda, gv + gu);
                a_next = att;
                Rsum = fma(double(gv + gu), double(rec.x), Rsum);
                kacc = fma(fma(double(rec.y), double(lambda), -Rsum), P.ds, kacc);
                --kk;
            } else {
                tau = fma(-double(kap), P.ds, tau);                               // tau_k = tau_{k+1} - kappa_k ds
                const float T = ex2_approx(float(tau * -1.4426950408889634));     // exp(-tau_k)
                lambda = fmaf(a_next, lambda, (gv + gu) * P.emis);                // lambda_{k+1} ds
                a_next = att;
                const float v = lambda * T;
#pragma unroll
                for (int s = 0; s < 8; ++s) S.acc[s].v[0] = fmaf(w[s], v, S.acc[s].v[0]);
            }

            const int c0 = A[0].p.c, c1 = A[1].p.c, c2 = A[2].p.c;
#pragma unroll
            for (int a = 0; a < 3; ++a) fx_add(A[a].p, A[a].d);
            if ((c0 ^ A[0].p.c) | (c1 ^ A[1].p.c) | (c2 ^ A[2].p.c)) {
                if (P.ds_f >= 1.0f && (((A[0].p.c - c0) | (A[1].p.c - c1) | (A[2].p.c - c2)) > 1)) {
                    S.flush_all(og, A);
                    S.restart(P, A, negbits, bin, gs);
                } else {
                    if (c0 != A[0].p.c) S.template axis_step<0>(P, A, negbits, og, gs);
                    if (c1 != A[1].p.c) S.template axis_step<1>(P, A, negbits, og, gs);
                    if (c2 != A[2].p.c) S.template axis_step<2>(P, A, negbits, og, gs);
                }
                if (WRT_KAPPA) {                     // the kappa cell may have changed: reduce the old one's sum
                    const int ko_old = ko;
                    load_kappa();
                    if (ko != ko_old) {
                        if (kacc != 0.0)
                            asm volatile("red.global.add.f64 [%0], %1;" ::"l"(og + ko_old), "d"(kacc) : "memory");
                        kacc = 0.0;
                    }
                } else {
                    load_kappa();
                }
            }
        }
    }
    if (WRT_KAPPA) flush_kappa();
    else S.flush_all(og, A);
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
