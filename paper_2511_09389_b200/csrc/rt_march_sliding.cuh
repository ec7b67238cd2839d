// rt_march_sliding.cuh — the sliding stencil (sm_100a): register accumulation of the trilinear deposit, used by every
// march kernel, and march_sliding_kernel, the march without phases, weight table and scratch (round 1's product kernel:
// now the kernel of the rt_march_ex variants, of substeps of a cell or more and of the kappa adjoint's record pass).
//
// One thread marches one (source, direction, bin-group) ray for all n_steps * N_s substeps of eq. (2)
// (PAPER.md:23).  The 8 voxels of the ray's clamped trilinear stencil live in registers: their j
// values (read once per voxel) and their pending deposits.  A voxel's pending deposit is reduced to memory
// (red.global.add) only when the stencil slides off it, so a ray issues ~1 reduction per substep instead of 8,
// and a ray that has left the box on all three axes issues one reduction for the rest of its path.  The sums are
// the same sums (each voxel still receives every w_c I_{k+1}); only their association changes.
//
// TRAVEL COORDINATES.  Each axis is marched in a coordinate u that ascends: u = x on an ascending axis and, on a
// descending one, the bitwise complement of the fixed-point position, U = ~X = -X - 1, i.e. u = -x - 2^-64 (the
// increment is -D, exact).  A cell crossing is then always "the cell word of u went up", the stencil's slots are
// (trailing, leading) per axis, and a slide flushes the 4 trailing slots, moves 4, loads 4.  The grid point of
// u-cell c is array index c (ascending) or -c (descending).  With the complement (rather than the negation):
//   * floor(x) -- the nearest-neighbour kappa cell, PAPER.md:29 / D4 -- is ALWAYS the leading index of a
//     descending axis (and the trailing index of an ascending one), also when x sits exactly on a cell plane;
//   * on a plane x = m the u-fraction is all ones, so the leading weight rounds to exactly 1 and the trailing
//     one (~fraction = 0) to exactly 0: the same corners and weights as the array-coordinate stencil (m, m+1).
//
// WEIGHTS.  Leading weight f = top 32 fraction bits, trailing weight = their complement (each truncated to the
// 2^-32 grid, so tiny weights keep their relative accuracy); conversions stay unscaled (values up to 2^32) and
// the 2^-96 of the triple product is folded into the z pair.  CLAMPING (D5): where both indices of
// an axis clamp to the same voxel the two slots are merged -- the fraction is masked to 0, which makes the pair
// exactly (trailing 1, leading 0) -- and nothing slides while the ray moves on outside the box.
#pragma once
#include "rt_common.cuh"

namespace rt {

// accumulator / j-cache slot for (plane p of axis AX, other two axes u, v); slots are [x][y][z], 0 = trailing
template <int AX> __device__ __forceinline__ constexpr int slot(int p, int u, int v) {
    return AX == 0 ? (p * 4 + u * 2 + v) : (AX == 1 ? (u * 4 + p * 2 + v) : (u * 4 + v * 2 + p));
}

// number of slots in use below s (slots in use: those with no bit outside `bits`)
__host__ __device__ constexpr int slot_rank(int s, int bits) {
    int r = 0;
    for (int t = 0; t < s; ++t) r += ((t & ~bits) == 0) ? 1 : 0;
    return r;
}

__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

struct TravelAxis {
    Fx96 p, d;          // position and per-substep increment in travel coordinates (d >= 0)
    int dl;             // leading minus trailing element offset of this axis (0 = merged)
    uint32_t fmask;     // 0 while merged (dl == 0), else all ones
};

// element offset of u-cell c of axis AX (array index c, or -c on a descending axis, clamped: PAPER.md:29)
template <int AX> __device__ __forceinline__ int eoff(const MarchParams& P, int c, int negbits) {
    const int lim = (AX == 0 ? P.nx : (AX == 1 ? P.ny : P.nz)) - 1;
    const int stride = AX == 0 ? P.ny * P.nz * P.nb : (AX == 1 ? P.nz * P.nb : P.nb);
    const int idx = (negbits & (1 << AX)) ? -c : c;
    return min(max(idx, 0), lim) * stride;
}

// The stencil: 8 register slots [x][y][z], 0 = trailing / 1 = leading per axis.  Slot s sits at element offset
// base + (s&4 ? dl_x : 0) + (s&2 ? dl_y : 0) + (s&1 ? dl_z : 0); base includes the thread's bin offset.
// KTRI (D18): kappa is read trilinearly too, so its 8 corner values are cached like j's.
template <int NB, typename ACC, bool KTRI> struct Stencil {
    BinVec<NB> acc[8];   // pending deposits for the 8 stencil voxels
    BinVec<NB> jc[8];    // j at the 8 stencil voxels
    BinVec<NB> kc[KTRI ? 8 : 1];   // kappa at the 8 stencil voxels (trilinear-kappa variant only)
    int base;            // element offset of slot 0

    __device__ __forceinline__ int off(int s, const TravelAxis (&A)[3]) const {
        return base + ((s & 4) ? A[0].dl : 0) + ((s & 2) ? A[1].dl : 0) + ((s & 1) ? A[2].dl : 0);
    }
    __device__ __forceinline__ void flush_slot(ACC* og, int s, const TravelAxis (&A)[3]) {
        if (any_nonzero<NB>(acc[s])) red_bins(og + off(s, A), acc[s]);
    }
    __device__ __forceinline__ void zero_slot(int s) {
#pragma unroll
        for (int b = 0; b < NB; ++b) acc[s].v[b] = 0.0f;
    }
    // ACT (here and in axis_step): bit a set = axis a is ACTIVE.  An inactive axis is one every ray of the warp has
    // left the box through for good (march_phased_kernel's lower-dimensional phases): its leading slots hold exactly
    // zero and are skipped, i.e. only the slots whose index bit (4 >> a) is clear are touched.  ACT = 7: all 8 slots.
    template <int ACT = 7> __device__ __forceinline__ void flush_all(ACC* og, const TravelAxis (&A)[3]) {
        constexpr int kBits = ((ACT & 1) ? 4 : 0) | ((ACT & 2) ? 2 : 0) | ((ACT & 4) ? 1 : 0);
#pragma unroll
        for (int s = 0; s < 8; ++s)
            if ((s & ~kBits) == 0) {
                flush_slot(og, s, A);
                zero_slot(s);
            }
    }
    template <int AX> __device__ __forceinline__ int place(const MarchParams& P, TravelAxis& X, int negbits) {
        const int t = eoff<AX>(P, X.p.c, negbits);
        X.dl = eoff<AX>(P, X.p.c + 1, negbits) - t;
        X.fmask = X.dl ? 0xFFFFFFFFu : 0u;
        return t;
    }
    // (re)build the stencil at the axes' current cells; pending deposits must have been flushed
    __device__ __forceinline__ void restart(const MarchParams& P, TravelAxis (&A)[3], int negbits, int bin_off,
                                            const float* jsrc) {
        base = bin_off + place<0>(P, A[0], negbits) + place<1>(P, A[1], negbits) + place<2>(P, A[2], negbits);
        reload(P, A, jsrc);
    }
    // (re)read the cached values of the 8 stencil voxels from `jsrc`
    __device__ __forceinline__ void reload(const MarchParams& P, const TravelAxis (&A)[3], const float* jsrc) {
#pragma unroll
        for (int s = 0; s < 8; ++s) {
            jc[s] = ld_bins<NB>(jsrc + off(s, A));
            if constexpr (KTRI) kc[s] = ld_bins<NB>(P.kappa + off(s, A));
        }
    }
    // Axis AX advanced by one cell.  The old leading plane is the new trailing plane (also under clamping: both
    // are clamp(c+1)), so the trailing index moves iff the axis was not merged; the new leading index is looked up.
    // flush_plane() reduces the pending sums of the trailing plane of AX to memory (called before anything moves, with
    // base / dl still those of the old stencil; the cell word of AX may already be the new one).
    template <int AX, int ACT = 7, class FlushPlane>
    __device__ __forceinline__ void axis_step_with(const MarchParams& P, TravelAxis (&A)[3], int negbits, const float* jsrc,
                                                   FlushPlane&& flush_plane) {
        constexpr int kBits = ((ACT & 1) ? 4 : 0) | ((ACT & 2) ? 2 : 0) | ((ACT & 4) ? 1 : 0);
        TravelAxis& X = A[AX];
        // new leading minus new trailing offset: +-stride while both indices are inside the domain, i.e. u-cell
        // c in [0, lim-1] (ascending: indices c, c+1) or [-lim, -1] (descending: indices -c, -c-1); else 0
        const int lim = (AX == 0 ? P.nx : (AX == 1 ? P.ny : P.nz)) - 1;
        const int stride = AX == 0 ? P.ny * P.nz * P.nb : (AX == 1 ? P.nz * P.nb : P.nb);
        const bool neg = (negbits & (1 << AX)) != 0;
        const bool inside = uint32_t(X.p.c + (neg ? lim : 0)) < uint32_t(lim);
        const int dln = inside ? (neg ? -stride : stride) : 0;
        const bool move = (X.dl != 0), load = inside;
        if (move) {
            flush_plane();
#pragma unroll
            for (int u = 0; u < 2; ++u)
#pragma unroll
                for (int v = 0; v < 2; ++v) {
                    const int s0 = slot<AX>(0, u, v), s1 = slot<AX>(1, u, v);
                    if (s1 & ~kBits) continue;       // a slot on the leading side of an inactive axis
                    acc[s0] = acc[s1];
                    jc[s0] = jc[s1];
                    if constexpr (KTRI) kc[s0] = kc[s1];
                    zero_slot(s1);
                }
        }
        base += X.dl;                 // the trailing index becomes the old leading one (dl = 0 when nothing moved)
        X.dl = dln;
        X.fmask = inside ? 0xFFFFFFFFu : 0u;
        if (load) {
#pragma unroll
            for (int u = 0; u < 2; ++u)
#pragma unroll
                for (int v = 0; v < 2; ++v) {
                    const int s1 = slot<AX>(1, u, v);
                    if (s1 & ~kBits) continue;
                    jc[s1] = ld_bins<NB>(jsrc + off(s1, A));
                    if constexpr (KTRI) kc[s1] = ld_bins<NB>(P.kappa + off(s1, A));
                }
        }
    }
    // The slide with the loads DEFERRED: the new leading plane is only marked in `stale` (bit s = slot s must be read
    // again), a moved slot takes its mark along, and load_stale() reads every marked slot once all the axes that
    // crossed in this substep have slid.  The register moves of a later slide then never wait for an earlier slide's
    // loads (one L2 round trip per substep instead of up to three), and a double / triple crossing reads 6 / 7
    // voxels instead of 8 / 12.
    template <int AX, int ACT = 7, class FlushPlane>
    __device__ __forceinline__ void axis_slide_deferred(const MarchParams& P, TravelAxis (&A)[3], int negbits, uint32_t& stale,
                                                        FlushPlane&& flush_plane) {
        constexpr int kBits = ((ACT & 1) ? 4 : 0) | ((ACT & 2) ? 2 : 0) | ((ACT & 4) ? 1 : 0);
        constexpr int kAxBit = AX == 0 ? 4 : (AX == 1 ? 2 : 1);
        uint32_t lead = 0;               // mask of the slots in use on the leading side of AX
        for (int t = 0; t < 8; ++t)
            if ((t & kAxBit) && !(t & ~kBits)) lead |= 1u << t;
        TravelAxis& X = A[AX];
        const int lim = (AX == 0 ? P.nx : (AX == 1 ? P.ny : P.nz)) - 1;
        const int stride = AX == 0 ? P.ny * P.nz * P.nb : (AX == 1 ? P.nz * P.nb : P.nb);
        const bool neg = (negbits & (1 << AX)) != 0;
        const bool inside = uint32_t(X.p.c + (neg ? lim : 0)) < uint32_t(lim);
        const int dln = inside ? (neg ? -stride : stride) : 0;
        if (X.dl != 0) {
            flush_plane();
#pragma unroll
            for (int u = 0; u < 2; ++u)
#pragma unroll
                for (int v = 0; v < 2; ++v) {
                    const int s0 = slot<AX>(0, u, v), s1 = slot<AX>(1, u, v);
                    if (s1 & ~kBits) continue;
                    acc[s0] = acc[s1];
                    jc[s0] = jc[s1];
                    if constexpr (KTRI) kc[s0] = kc[s1];
                    zero_slot(s1);
                }
            stale = (stale & ~(lead | (lead >> kAxBit))) | ((stale & lead) >> kAxBit);
        }
        base += X.dl;
        X.dl = dln;
        X.fmask = inside ? 0xFFFFFFFFu : 0u;
        if (inside) stale |= lead;
    }
    template <int ACT = 7>
    __device__ __forceinline__ void load_stale(const MarchParams& P, const TravelAxis (&A)[3], const float* jsrc, uint32_t stale) {
        constexpr int kBits = ((ACT & 1) ? 4 : 0) | ((ACT & 2) ? 2 : 0) | ((ACT & 4) ? 1 : 0);
#pragma unroll
        for (int s = 0; s < 8; ++s)
            if (!(s & ~kBits) && ((stale >> s) & 1u)) {
                jc[s] = ld_bins<NB>(jsrc + off(s, A));
                if constexpr (KTRI) kc[s] = ld_bins<NB>(P.kappa + off(s, A));
            }
    }
    // the trailing plane of AX reduced slot by slot into the accumulation grid `og`
    template <int AX, int ACT = 7> __device__ __forceinline__ void flush_trailing(ACC* og, const TravelAxis (&A)[3]) {
        constexpr int kBits = ((ACT & 1) ? 4 : 0) | ((ACT & 2) ? 2 : 0) | ((ACT & 4) ? 1 : 0);
#pragma unroll
        for (int u = 0; u < 2; ++u)
#pragma unroll
            for (int v = 0; v < 2; ++v) {
                if (slot<AX>(1, u, v) & ~kBits) continue;
                flush_slot(og, slot<AX>(0, u, v), A);
            }
    }
    // the slide with the trailing plane reduced slot by slot into the accumulation grid `og`
    template <int AX, int ACT = 7>
    __device__ __forceinline__ void axis_step(const MarchParams& P, TravelAxis (&A)[3], int negbits, ACC* og,
                                              const float* jsrc) {
        constexpr int kBits = ((ACT & 1) ? 4 : 0) | ((ACT & 2) ? 2 : 0) | ((ACT & 4) ? 1 : 0);
        axis_step_with<AX, ACT>(P, A, negbits, jsrc, [&]() {
#pragma unroll
            for (int u = 0; u < 2; ++u)
#pragma unroll
                for (int v = 0; v < 2; ++v) {
                    if (slot<AX>(1, u, v) & ~kBits) continue;
                    flush_slot(og, slot<AX>(0, u, v), A);
                }
        });
    }
};

// STEP: the rt_march_step form -- start at substep P.k0 with (I, exp(-tau)) loaded from the ray state, store them back
// RECORD (rt_march_adjoint_kappa): nothing is deposited; I_{k+1}, scaled by 4 pi/N_Omega, of every substep goes to
// record[k * record_stride + thread], a warp writing one 128-byte run per substep.
// COPIES: block b reduces into copy b % P.acc_copies of the accumulation grid.  ncu shows this march loading the L2
// slices unevenly (atomic input 19-67 % busy across slices: the voxels next to the sources and on the faces are
// hot); a few copies of a small grid spread a hot voxel over as many addresses, snapshot_finalize_kernel adds them
// up (C2: 18.1 -> 17.2 ms with 3 copies).  A separate instantiation: the plain kernel's code stays as it is.
template <int NB, typename ACC, int MINB, bool STEP, bool KTRI = false, bool RECORD = false, bool COPIES = false>
__global__ void __launch_bounds__(kThreads, MINB) march_sliding_kernel(const MarchParams P, float* record = nullptr,
                                                                       long long record_stride = 0) {
    if constexpr (COPIES)
        if (P.same_frac && *P.same_frac) return;     // (unused since the phased kernel took over the weight table)
    // the batched path launches the next batch (other scratch grid, no dependence on this one) with programmatic
    // stream serialization: it may start as soon as every block of this grid has started, filling this grid's tail
    // (and waits for this grid's completion at its own end: griddepcontrol.wait below)
    if constexpr (NB == 4) asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    RayId id;
    if (!ray_id(P, id)) return;
    ACC* og = static_cast<ACC*>(P.acc);      // the bin offset id.group * NB rides in the stencil's base offset
    if constexpr (COPIES) og += (blockIdx.x % unsigned(P.acc_copies)) * P.acc_copy_stride;

    TravelAxis A[3];
    int negbits = 0;                         // bit a: the ray descends axis a
    {
        double nh[3];
        fib_direction(id.index, uint32_t(P.n_rays), nh);
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const bool neg = nh[a] < 0.0;
            A[a].p = fx_from_double(source_coord(P, id.src, a), neg ? kFxComplement : kFxPlain);
            A[a].d = fx_from_double(__dmul_rn(P.ds, nh[a]), neg ? kFxNegate : kFxPlain);
            negbits |= neg ? (1 << a) : 0;
            if (STEP) fx_advance(A[a].p, A[a].d, P.k0);      // x_k0 = x_0 + k0 ds n
        }
    }
    asm volatile("" : "+r"(negbits));        // opaque: keeps ptxas from re-deriving the signs with fp64 compares
    Stencil<NB, ACC, KTRI> S;
#pragma unroll
    for (int s = 0; s < 8; ++s) S.zero_slot(s);
    S.restart(P, A, negbits, id.group * NB, P.j);

    float I[NB], T[NB], att[NB];     // I scaled by 4 pi/N_Omega; T = exp(-tau); att = exp(-kappa ds) of the kappa cell
#pragma unroll
    for (int b = 0; b < NB; ++b) { I[b] = 0.0f; T[b] = 1.0f; }
    const size_t state_at = (size_t(id.src) * P.n_rays + id.index) * P.nb + size_t(id.group) * NB;
    if (STEP) {                        // the ray's (I, exp(-tau)) carried from the previous call
        const BinVec<NB> si = ld_bins<NB>(P.state_I + state_at), sT = ld_bins<NB>(P.state_T + state_at);
#pragma unroll
        for (int b = 0; b < NB; ++b) { I[b] = si.v[b]; T[b] = sT.v[b]; }
    }
    // kappa: nearest neighbour at clamp(floor(x_k)) (D4) = trailing index, leading on descending axes
    auto load_att = [&]() {
        const int ko = S.base + ((negbits & 1) ? A[0].dl : 0) + ((negbits & 2) ? A[1].dl : 0) + ((negbits & 4) ? A[2].dl : 0);
        const BinVec<NB> kap = ld_bins<NB>(P.kappa + ko);
#pragma unroll
        for (int b = 0; b < NB; ++b) att[b] = ex2_approx(kap.v[b] * P.att_scale);
    };
    if (!KTRI) load_att();
    const bool long_steps = !(P.ds_f < 1.0f);      // only then can one substep cross more than one cell plane

    for (int m = 0; m < P.n_steps; ++m) {
        for (int k = 0; k < P.n_sub; ++k) {
            // unscaled weights in [0, 2^32]; 2^-96 rides on the z pair
            const uint32_t hx = A[0].p.fh & A[0].fmask, hy = A[1].p.fh & A[1].fmask, hz = A[2].p.fh & A[2].fmask;
            const float lx = __uint2float_rn(hx), tx = __uint2float_rn(~hx);
            const float ly = __uint2float_rn(hy), ty = __uint2float_rn(~hy);
            const float wz[2] = {__uint2float_rn(~hz) * 1.2621774483536189e-29f,      // 2^-96
                                 __uint2float_rn(hz) * 1.2621774483536189e-29f};
            const float wxy[4] = {tx * ty, tx * ly, lx * ty, lx * ly};
            float w[8];
            float jv[NB], ju[NB];          // two partial sums: half the dependent-FMA chain length
#pragma unroll
            for (int s = 0; s < 8; ++s) w[s] = wxy[s >> 1] * wz[s & 1];
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                jv[b] = w[0] * S.jc[0].v[b];
                ju[b] = w[1] * S.jc[1].v[b];
            }
#pragma unroll
            for (int s = 2; s < 8; s += 2)
#pragma unroll
                for (int b = 0; b < NB; ++b) {
                    jv[b] = fmaf(w[s], S.jc[s].v[b], jv[b]);
                    ju[b] = fmaf(w[s + 1], S.jc[s + 1].v[b], ju[b]);
                }
#pragma unroll
            for (int b = 0; b < NB; ++b) jv[b] += ju[b];
            if constexpr (KTRI) {          // kappa(x_k) with the weights of j(x_k); one exponential per substep
#pragma unroll
                for (int b = 0; b < NB; ++b) {
                    float kv = 0.0f;
#pragma unroll
                    for (int s = 0; s < 8; ++s) kv = fmaf(w[s], S.kc[s].v[b], kv);
                    att[b] = ex2_approx(kv * P.att_scale);
                }
            }
#pragma unroll
            for (int b = 0; b < NB; ++b) {                       // eq. (2)
                const float emitted = jv[b] * T[b] * P.emis;
                I[b] = fmaf(I[b], att[b], emitted);
                T[b] *= att[b];
                if (RECORD && b == 0)
                    record[((long long)m * P.n_sub + k) * record_stride + (long long)blockIdx.x * kThreads + threadIdx.x] =
                        I[0];
            }
            if (!RECORD) {
#pragma unroll
                for (int s = 0; s < 8; ++s)
#pragma unroll
                    for (int b = 0; b < NB; ++b) S.acc[s].v[b] = fmaf(w[s], I[b], S.acc[s].v[b]);
            }

            // x_{k+1} = x_k + n ds; a changed cell word is a crossing (increments are >= 0 in travel coordinates)
            const int c0 = A[0].p.c, c1 = A[1].p.c, c2 = A[2].p.c;
#pragma unroll
            for (int a = 0; a < 3; ++a) fx_add(A[a].p, A[a].d);
            if ((c0 ^ A[0].p.c) | (c1 ^ A[1].p.c) | (c2 ^ A[2].p.c)) {
                if (long_steps && (((A[0].p.c - c0) | (A[1].p.c - c1) | (A[2].p.c - c2)) > 1)) {
                    S.flush_all(og, A);            // a step longer than a cell: restart the stencil
                    S.restart(P, A, negbits, id.group * NB, P.j);
                } else {
                    if (c0 != A[0].p.c) S.template axis_step<0>(P, A, negbits, og, P.j);
                    if (c1 != A[1].p.c) S.template axis_step<1>(P, A, negbits, og, P.j);
                    if (c2 != A[2].p.c) S.template axis_step<2>(P, A, negbits, og, P.j);
                }
                if (!KTRI) load_att();
            }
        }
        S.flush_all(og, A);    // time-step boundary: the increments of step m are complete (rays continue, D7)
        og += P.snap_stride;
    }
    if (STEP) {
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            P.state_I[state_at + b] = I[b];
            P.state_T[state_at + b] = T[b];
        }
    }
    // A grid launched with programmatic stream serialization (the second batch of a pair) must not COMPLETE before
    // its prerequisite grid has: the drain_kernel that follows is ordered behind this grid only.  The wait comes
    // last, so the overlap is kept (this grid's tail is later than the first grid's anyway); it returns at once in a
    // normally launched grid.
    if constexpr (NB == 4) asm volatile("griddepcontrol.wait;" ::: "memory");
}

}  // namespace rt
