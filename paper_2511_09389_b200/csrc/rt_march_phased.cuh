// rt_march_phased.cuh — the product march kernel of rt_march (sm_100a): the sliding-stencil march of
// rt_march_sliding.cuh in warp-uniform PHASES, depositing into an fp32 scratch grid that is drained into the fp64
// accumulation grid while the march runs.
//
// One thread marches one (source, direction, bin group) ray through all n_steps * N_s substeps of eq. (2)
// with the clamped trilinear stencil of PAPER.md:29 held in registers (Stencil, rt_march_sliding.cuh).
//
// PHASES.  ACT = set of ACTIVE axes (bit a).  An axis becomes inactive once EVERY ray of the warp has left the box
// through it for good -- travel-coordinate cell word beyond the far face; cell words only go up, so the axis stays
// merged (rt_march_sliding.cuh) for the rest of the march: its leading weight is 0 and its trailing weight 1 in every
// lane.  The rays of a warp are neighbours (32 sorted sources x 1 direction, or 32 neighbouring directions of one
// source), so they leave through the same faces at about the same time (C2: of 444 substeps a warp spends 148 with
// three active axes, 158 with two, 112 with one, 26 with none; 74 % of C2's ray-substeps lie outside the box, where
// the paper's clamped deposits continue).  phase<ACT> is the substep loop with the inactive axes
// compiled out: 2^n stencil slots (weights, gather, deposit), position advance, slides and crossing tests for the n
// active axes only -- the same sums without the terms that are exactly zero.  It returns the next set of active axes
// (a warp vote after a cell crossing).  This is a restructuring, not a cut-off: every substep of every ray is taken.
//
// TABLE.  With sources that share their cell fractions (cell-centred sources; C2, C3) and a warp of
// 32 sources x ONE direction, the fraction words and crossing flags are the same in every lane: every 32 substeps
// lane l evaluates substep g + l -- x_{g+l} = x_0 + (g + l) ds n in the 96-bit fixed-point arithmetic of D3 -- into a
// 1 KB shared-memory table of per-axis (trailing, leading) weight pairs, the crossing flag in the sign bit of the
// trailing weight; a lane keeps only its cell words.  Whether the sources qualify is decided on the device
// (same_fraction_kernel); the TABLE and the plain instantiation are both launched and one returns at once.
//
// DEPOSITS.  One bin per thread: the fp32 window-brick scratch of rt_brick.cuh (one vector reduction per stencil
// plane).  Four bins per thread: the scratch is the plain [x][y][z][bin] grid and a voxel's four bins are one
// red.global.add.v4.f32.  Either way every block drains a slice of the scratch into the fp64 grid when its rays are
// done (rt_brick.cuh): no fp32 sum holds more than a fraction of the rays, and there are no batch boundaries.
#pragma once
#include "rt_brick.cuh"
#include "rt_march_sliding.cuh"

namespace rt {

// flag = 1 iff ds < 1 and every source has the fractional cell offsets of source 0 -- compared as the 64 fraction
// bits of the fixed-point coordinates the kernels march with (exact; float arithmetic on x - floor(x) would round
// e.g. -1e-10 and -3e-10 to the same 1.0f)
__global__ void same_fraction_kernel(int* flag, const float* sources, int n_src, float ds) {
    __shared__ int differs;
    if (threadIdx.x == 0) differs = (ds < 1.0f) ? 0 : 1;      // a substep of a cell or more may cross two planes
    __syncthreads();
    int bad = 0;
    for (int s = threadIdx.x; s < n_src; s += blockDim.x)
        for (int a = 0; a < 3; ++a) {
            const float x = sources[3 * size_t(s) + a], x0 = sources[a];
            const Fx96 p = fx_from_double(double(fminf(fmaxf(x, -536870912.0f), 536870912.0f)));
            const Fx96 p0 = fx_from_double(double(fminf(fmaxf(x0, -536870912.0f), 536870912.0f)));
            bad |= (p.fh != p0.fh) | (p.fl != p0.fl) | !(x == x);      // a NaN coordinate: leave it to the plain kernel
        }
    if (bad) atomicOr(&differs, 1);
    __syncthreads();
    if (threadIdx.x == 0) *flag = differs ? 0 : 1;
}

struct TableRow {            // substep g of a direction: 32 bytes = three (trailing, leading) weight pairs
    float t[3][2];           // per axis: float(~h) 2^-32, float(h) 2^-32 of the top 32 fraction bits h of x_g (travel
    int pad[2];              // coordinates, rt_march_sliding.cuh).  The SIGN BIT of the trailing weight is the
};                           // crossing flag of the axis: the cell word goes up between x_g and x_{g+1}

// (t, l) of an axis with the clamping mask of the lane applied: m = ~0 leaves the pair, m = 0 -- both
// indices of the axis clamp to one voxel -- makes it exactly (1, 0).  The same values as masking the fraction word
// before the conversions.  The sign bit of t (crossing flag) is dropped by the caller's fabsf.
__device__ __forceinline__ void mask_pair(float& t, float& l, uint32_t m) {
    t = __uint_as_float((__float_as_uint(t) & m) | (0x3F800000u & ~m));
    l = __uint_as_float(__float_as_uint(l) & m);
}

// The state one lane carries through the march
template <int NB, typename ACC = float, bool JVP = false, bool KTRI = false> struct PhasedLane {
    Stencil<NB, ACC, KTRI> S;
    TravelAxis A[3];         // TABLE: only the cell word, dl and fmask are used
    float I[NB], T[NB], att[NB];   // I scaled by 4 pi/N_Omega; T = exp(-tau) ds 4 pi/N_Omega; att = exp(-kappa ds) of the kappa cell
                                   // (kappa itself in the instantiations that convert per substep, phased_load_att)
    float Id[JVP ? NB : 1], Td[JVP ? NB : 1], u[JVP ? NB : 1];     // JVP (D21): tangents of I and T, and dkappa ds of the kappa cell
    ACC* sg;                 // scratch (fp64 grid if ACC = double) of the current time step
    int woff;                // NB == 1: float offset in it of the window the trailing slots start (rt_brick.cuh)
    int g;                   // substep index since x_0
    int left;                // substeps left in the current time step
    uint32_t roff;           // TABLE: byte offset of the row of substep g in the warp's table
    long long rec_at;        // RECORD: the thread's column of the record, or -1 for a lane without a ray of its own
};

// array index of u-cell c of axis AX (c, or -c on a descending axis), clamped to the grid
template <int AX> __device__ __forceinline__ int aidx(const MarchParams& P, int c, int negbits) {
    const int lim = (AX == 0 ? P.nx : (AX == 1 ? P.ny : P.nz)) - 1;
    return min(max((negbits & (1 << AX)) ? -c : c, 0), lim);
}

// The pending sums of the lane's stencil as brick payloads (rt_brick.cuh; one bin per thread).  Slots are [x][y][z]
// roles, 0 = trailing / 1 = leading in TRAVEL order; a brick is in ARRAY order, so on a descending axis the leading
// slot is the lower element.  The lower index of an axis is (trailing index - 1 on a descending axis), also when the
// axis is merged: the other element of the pair is then padding or a neighbour and carries the leading slot's exact
// zero.  Slots on the leading side of an inactive axis (ACT) do not exist: zero.
template <int ACT, class STENCIL> struct BrickView {
    const STENCIL& S;
    bool ny, nz;             // the ray descends y / z
    __device__ __forceinline__ float val(int rx, int ry, int rz) const {
        if ((rx && !(ACT & 1)) || (ry && !(ACT & 2)) || (rz && !(ACT & 4))) return 0.0f;
        return S.acc[rx * 4 + ry * 2 + rz].v[0];
    }
    // element (iy, iz) of the 2 x 2 (y, z) window of x slot rx, array order
    __device__ __forceinline__ void window(int rx, float (&e)[2][2]) const {
        float z0[2], z1[2];      // per y ROLE: lower / upper z element
#pragma unroll
        for (int ry = 0; ry < 2; ++ry) {
            z0[ry] = nz ? val(rx, ry, 1) : val(rx, ry, 0);
            z1[ry] = nz ? val(rx, ry, 0) : val(rx, ry, 1);
        }
        e[0][0] = ny ? z0[1] : z0[0]; e[0][1] = ny ? z1[1] : z1[0];
        e[1][0] = ny ? z0[0] : z0[1]; e[1][1] = ny ? z1[0] : z1[1];
    }
};

// Reduce the trailing plane of axis AX into the brick scratch and move the lane's window offset along with the
// stencil.  Called from Stencil::axis_step_with before the stencil moves, i.e. only when the trailing index of AX
// really changes (by +1 ascending, -1 descending).  AX = -1: all planes, nothing moves (time-step boundary).
// L.woff is the window that starts at (lower y index, lower z index) of the trailing x slot; the leading x slot is one
// x step on (if x is merged its sums are exact zeros and nothing is issued); a y-slide uses the window that starts at
// the trailing row itself, a z-slide the one that starts at the trailing column.
template <int AX, int ACT, class LANE>
__device__ __forceinline__ void brick_flush(const BrickGeom& G, LANE& L, int negbits) {
    const BrickView<ACT, decltype(L.S)> V{L.S, (negbits & 2) != 0, (negbits & 4) != 0};
    const int dx = (negbits & 1) ? -G.sx : G.sx;
    float* w0 = L.sg + L.woff;
    float e[2][2];
    if (AX == 0 || AX == -1) {               // the (y, z) window of the trailing x slot: one brick
        V.window(0, e);
        red_v4(w0, e[0][0], e[0][1], e[1][0], e[1][1]);
    }
    if (AX == -1 && (ACT & 1)) {             // ... and of the leading x slot
        V.window(1, e);
        red_v4(w0 + dx, e[0][0], e[0][1], e[1][0], e[1][1]);
    }
    if (AX == 1) {                           // the z pair of the trailing y row, per x slot
#pragma unroll
        for (int rx = 0; rx < ((ACT & 1) ? 2 : 1); ++rx) {
            const float lo = V.nz ? V.val(rx, 0, 1) : V.val(rx, 0, 0), hi = V.nz ? V.val(rx, 0, 0) : V.val(rx, 0, 1);
            red_v2(w0 + (rx ? dx : 0) + (V.ny ? G.sy : 0), lo, hi);
        }
    }
    if (AX == 2) {                           // the y pair of the trailing z column, per x slot: elements 0 and 2 of a brick
#pragma unroll
        for (int rx = 0; rx < ((ACT & 1) ? 2 : 1); ++rx) {
            const float lo = V.ny ? V.val(rx, 1, 0) : V.val(rx, 0, 0), hi = V.ny ? V.val(rx, 0, 0) : V.val(rx, 1, 0);
            red_v4(w0 + (rx ? dx : 0) + (V.nz ? 4 : 0), lo, 0.0f, hi, 0.0f);
        }
    }
    if (AX == 0) L.woff += dx;
    if (AX == 1) L.woff += V.ny ? -G.sy : G.sy;
    if (AX == 2) L.woff += V.nz ? -4 : 4;
}

// One stencil slide of the lane along axis AX, the trailing plane reduced into the scratch; the loads of the new
// leading plane are left to Stencil::load_stale (rt_march_sliding.cuh)
template <int AX, int ACT, bool BRICK, bool RECORD, class LANE>
__device__ __forceinline__ void phased_axis_step(const MarchParams& P, const BrickGeom& G, LANE& L, int negbits, uint32_t& stale) {
#ifdef RT_NO_DEFER
    if constexpr (BRICK)
        L.S.template axis_step_with<AX, ACT>(P, L.A, negbits, P.j, [&]() { brick_flush<AX, ACT>(G, L, negbits); });
    else
        L.S.template axis_step<AX, ACT>(P, L.A, negbits, L.sg, P.j);        // per voxel: one red.v4.f32 (red.f32) of its bins
#else
    if constexpr (RECORD)      // nothing is deposited, so nothing is flushed
        L.S.template axis_slide_deferred<AX, ACT>(P, L.A, negbits, stale, []() {});
    else if constexpr (BRICK)
        L.S.template axis_slide_deferred<AX, ACT>(P, L.A, negbits, stale, [&]() { brick_flush<AX, ACT>(G, L, negbits); });
    else      // per voxel: one red.v4.f32 (red.f32, red.f64 per bin) of its bins
        L.S.template axis_slide_deferred<AX, ACT>(P, L.A, negbits, stale, [&]() { L.S.template flush_trailing<AX, ACT>(L.sg, L.A); });
#endif
}

// kappa of the cell the lane is in (and dkappa of it, JVP).  RAW: the values are kept as loaded and turned into
// exp(-kappa ds) (dkappa ds) where a substep uses them -- in the instantiations whose lanes cross cell planes on their
// own the conversion right here would wait for the load in every substep (ncu: the top stall of the chunked march)
template <int NB, bool JVP, bool RAW, class LANE>
__device__ __forceinline__ void phased_load_att(const MarchParams& P, LANE& L, int ko) {
    const BinVec<NB> kap = ld_bins<NB>(P.kappa + ko);
#pragma unroll
    for (int b = 0; b < NB; ++b) L.att[b] = RAW ? kap.v[b] : ex2_approx(kap.v[b] * P.att_scale);
    if constexpr (JVP) {
        const BinVec<NB> dk = ld_bins<NB>(P.dkappa + ko);
#pragma unroll
        for (int b = 0; b < NB; ++b) L.u[b] = RAW ? dk.v[b] : dk.v[b] * P.ds_f;
    }
}

// The substep loop with the axes in ACT active; runs until the table runs out (TABLE), the time step ends or an
// axis goes inactive, and returns the new set of active axes.
template <int ACT, int NB, bool TABLE, bool BRICK, bool STEP, bool JVP, bool KTRI, bool RECORD, class LANE>
__device__ __forceinline__ int phase(const MarchParams& P, const BrickGeom& G, LANE& L, int negbits, uint32_t tbase) {
    constexpr int kBits = ((ACT & 1) ? 4 : 0) | ((ACT & 2) ? 2 : 0) | ((ACT & 4) ? 1 : 0);      // slot index bits in use
    constexpr int kActive = ((ACT & 1) ? 1 : 0) + ((ACT & 2) ? 1 : 0) + ((ACT & 4) ? 1 : 0);
    constexpr int kLast = (ACT & 4) ? 2 : ((ACT & 2) ? 1 : 0);                                   // the last active axis
    constexpr bool RAW = !TABLE && !KTRI;      // L.att holds kappa itself (phased_load_att)
    // Four bins per thread, lanes crossing on their own (the sorted march of large grids): the kappa load of a crossing goes
    // ahead of its slides (C4 13.65 -> 13.3 ms; the one-bin kernels lose 4-10 % to the extra arithmetic, C3 is unchanged)
    constexpr bool kEarlyKappa = NB == 4 && !TABLE && !KTRI;
    int next = ACT;
    do {
        float w[8];
        bool cross[3] = {false, false, false};
        if constexpr (ACT != 0) {
            float t[3] = {1.0f, 1.0f, 1.0f}, l[3] = {0.0f, 0.0f, 0.0f};
            if constexpr (TABLE) {
#pragma unroll
                for (int a = 0; a < 3; ++a)
                    if (ACT & (1 << a)) {
                        asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(t[a]), "=f"(l[a]) : "r"(tbase + L.roff + 8u * a));
                        // (the same in every lane; the vote makes it a uniform predicate, and the branches on it uniform: no
                        // reconvergence bookkeeping around the slides -- C2 12.08 -> 11.85 ms, C3 5.29 -> 5.06)
                        cross[a] = __any_sync(0xFFFFFFFFu, __float_as_int(t[a]) < 0);
                        mask_pair(t[a], l[a], L.A[a].fmask);
                        t[a] = fabsf(t[a]);
                    }
                L.roff = (L.roff + 32u) & 1023u;
            } else {
                // unscaled weights in [0, 2^32] from the lane's own fraction words; 2^(-32 n) rides on the last active axis
#pragma unroll
                for (int a = 0; a < 3; ++a)
                    if (ACT & (1 << a)) {
                        const uint32_t h = L.A[a].p.fh & L.A[a].fmask;
                        const float sc = (a == kLast) ? (kActive == 3 ? 1.2621774483536189e-29f
                                                                      : (kActive == 2 ? 5.421010862427522e-20f : 2.3283064365386963e-10f))
                                                      : 1.0f;
                        t[a] = __uint2float_rn(~h) * sc;
                        l[a] = __uint2float_rn(h) * sc;
                        const int c = L.A[a].p.c;              // x_{k+1} = x_k + n ds; a changed cell word is a crossing
                        fx_add(L.A[a].p, L.A[a].d);
                        cross[a] = L.A[a].p.c != c;
                    }
            }
            // weights of the slots in use: products over the active axes (an inactive axis contributes the factor 1)
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
        } else {
            w[0] = 1.0f;
        }
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            float jv = 0.0f, ju = 0.0f;      // two partial sums over alternate slots: half the dependent-FMA chain length
            if constexpr (ACT == 0) {
                jv = L.S.jc[0].v[b];
            } else {
#pragma unroll
                for (int s = 0; s < 8; ++s)
                    if ((s & ~kBits) == 0) {
                        const int r = slot_rank(s, kBits);       // position of s among the slots in use
                        const float jc = L.S.jc[s].v[b];
                        if (r & 1) ju = (r == 1) ? w[s] * jc : fmaf(w[s], jc, ju);
                        else jv = (r == 0) ? w[s] * jc : fmaf(w[s], jc, jv);
                    }
            }
            if constexpr (KTRI) {            // D18: kappa(x_k) with the weights of j(x_k); one exponential per substep and bin
                float kv = 0.0f;
                if constexpr (ACT == 0) {
                    kv = L.S.kc[0].v[b];
                } else {
#pragma unroll
                    for (int s = 0; s < 8; ++s)
                        if ((s & ~kBits) == 0) kv = (slot_rank(s, kBits) == 0) ? w[s] * L.S.kc[s].v[b] : fmaf(w[s], L.S.kc[s].v[b], kv);
                }
                L.att[b] = ex2_approx(kv * P.att_scale);
            }
            const float att = RAW ? ex2_approx(L.att[b] * P.att_scale) : L.att[b];
            if constexpr (JVP) {
                // the tangent of eq. (2) for kappa -> kappa + eps dkappa (D21), u = dkappa_k ds:
                //   Idot_{k+1} = a_k (Idot_k - I_k u) + J_k Tdot_k,   Tdot_{k+1} = a_k (Tdot_k - T_k u)      (old I, T on the right)
                const float u = RAW ? L.u[b] * P.ds_f : L.u[b];
                L.Id[b] = fmaf(att, fmaf(-L.I[b], u, L.Id[b]), (jv + ju) * L.Td[b]);
                L.Td[b] = att * fmaf(-L.T[b], u, L.Td[b]);
            }
            // eq. (2).  STEP: T is the carried exp(-tau) itself, else ds 4 pi/N_Omega rides on it
            const float emitted = STEP ? (jv + ju) * L.T[b] * P.emis : (jv + ju) * L.T[b];
            L.I[b] = fmaf(L.I[b], att, emitted);
            L.T[b] *= att;
            if constexpr (RECORD) {          // I_{k+1} of this substep; a warp writes one 128-byte run
                if (b == 0 && L.rec_at >= 0) P.record[(long long)L.g * P.record_stride + L.rec_at] = L.I[0];
            } else {
                const float dep = JVP ? L.Id[b] : L.I[b];       // what is deposited, with the weights of x_k
#pragma unroll
                for (int s = 0; s < 8; ++s)
                    if ((s & ~kBits) == 0)
                        L.S.acc[s].v[b] = (ACT == 0) ? L.S.acc[s].v[b] + dep : fmaf(w[s], dep, L.S.acc[s].v[b]);
            }
        }

        if constexpr (ACT != 0) {
            if (cross[0] | cross[1] | cross[2]) {     // TABLE: warp-uniform
                uint32_t stale = 0;
                if constexpr (kEarlyKappa) {
                    // the kappa cell AFTER the slides, worked out ahead of them (the arithmetic of Stencil::axis_slide_deferred
                    // without its moves): the load is issued before the reductions, moves and loads of the slides
                    int base = L.S.base, ko = 0;
#pragma unroll
                    for (int a = 0; a < 3; ++a)
                        if (ACT & (1 << a)) {
                            int dl = L.A[a].dl;
                            if (cross[a]) {
                                const int lim = (a == 0 ? P.nx : (a == 1 ? P.ny : P.nz)) - 1;
                                const int stride = a == 0 ? P.ny * P.nz * P.nb : (a == 1 ? P.nz * P.nb : P.nb);
                                const bool neg = (negbits & (1 << a)) != 0;
                                const bool inside = uint32_t(L.A[a].p.c + (neg ? lim : 0)) < uint32_t(lim);
                                base += dl;
                                dl = inside ? (neg ? -stride : stride) : 0;
                            }
                            ko += (negbits & (1 << a)) ? dl : 0;
                        }
                    phased_load_att<NB, JVP, RAW>(P, L, base + ko);
                }
#pragma unroll
                for (int a = 0; a < 3; ++a)
                    if ((ACT & (1 << a)) && cross[a]) {
                        if constexpr (TABLE) L.A[a].p.c += 1;
                        if (a == 0) phased_axis_step<0, ACT, BRICK, RECORD>(P, G, L, negbits, stale);
                        if (a == 1) phased_axis_step<1, ACT, BRICK, RECORD>(P, G, L, negbits, stale);
                        if (a == 2) phased_axis_step<2, ACT, BRICK, RECORD>(P, G, L, negbits, stale);
                        if constexpr (TABLE) {       // every lane crosses in the same substep: vote right here
                            const int lim = (a == 0 ? P.nx : (a == 1 ? P.ny : P.nz)) - 1;
                            const bool gone = L.A[a].p.c >= ((negbits & (1 << a)) ? 0 : lim);    // beyond the far face for good
                            if (__all_sync(0xFFFFFFFFu, gone)) next &= ~(1 << a);
                        }
                    }
                L.S.template load_stale<ACT>(P, L.A, P.j, stale);
                if constexpr (!KTRI && !kEarlyKappa) {
                    int ko = L.S.base;       // kappa: nearest neighbour at clamp(floor(x_k)) (D4)
                    if (ACT & 1) ko += (negbits & 1) ? L.A[0].dl : 0;
                    if (ACT & 2) ko += (negbits & 2) ? L.A[1].dl : 0;
                    if (ACT & 4) ko += (negbits & 4) ? L.A[2].dl : 0;
                    phased_load_att<NB, JVP, RAW>(P, L, ko);
                }
            }
            if constexpr (!TABLE) {
                if ((L.g & 7) == 7) {        // lanes cross at different substeps: vote every 8th substep
#pragma unroll
                    for (int a = 0; a < 3; ++a)
                        if (ACT & (1 << a)) {
                            const int lim = (a == 0 ? P.nx : (a == 1 ? P.ny : P.nz)) - 1;
                            const bool gone = L.A[a].p.c >= ((negbits & (1 << a)) ? 0 : lim);
                            if (__all_sync(0xFFFFFFFFu, gone)) next &= ~(1 << a);
                        }
                }
            }
        }
        ++L.g;
        --L.left;
    } while ((TABLE && ACT != 0 ? L.roff != 0 : true) && L.left != 0 && next == ACT);      // (no table without active axes)
    return next;
}

#ifndef RT_PHASED_MINB1
#define RT_PHASED_MINB1 8
#endif
#ifndef RT_PHASED_MINB1P
#define RT_PHASED_MINB1P 6
#endif
#ifndef RT_PHASED_MINB4
#define RT_PHASED_MINB4 4
#endif

// BRICK: the scratch is the window-brick grid of rt_brick.cuh (one-bin calls); else the plain grid [x][y][z][bin].
// ACC = double: no scratch -- the deposits are reduced straight into the fp64 grid (red.global.add.f64 per bin) and
// nothing is drained: for grids far larger than the L2, where a scratch would only add HBM traffic.
// STEP: the rt_march_step form (D17) -- one time step from substep P.k0, (I, exp(-tau)) of every ray loaded
// from and stored back to the ray state.
// JVP: the rt_march_jvp_kappa form (D21) -- the tangent of I for kappa -> kappa + eps P.dkappa is carried
// next to I and deposited instead of it.
// KTRI: the rt_march_trilinear_kappa form (D18) -- kappa cached at the stencil voxels like j and read with
// the trilinear weights every substep.
// ONE_DIR: every warp marches ONE direction (map_src = 1: 32 sources x 1 direction; always so with TABLE).
// RECORD: the first pass of rt_march_adjoint_kappa (D19) -- nothing is deposited; I_{k+1} of every
// substep go to P.record for the backward march (rt_adjoint.cuh), which maps its threads to rays the same way.
template <int NB, bool TABLE, bool BRICK = (NB == 1), typename ACC = float, bool STEP = false, bool JVP = false, bool KTRI = false,
          bool RECORD = false, bool ONE_DIR = TABLE>
__global__ void __launch_bounds__(kThreads, NB == 1 ? (TABLE ? RT_PHASED_MINB1 : RT_PHASED_MINB1P) : RT_PHASED_MINB4)
march_phased_kernel(const MarchParams P) {
    static_assert(!BRICK || (NB == 1 && sizeof(ACC) == 4), "the brick scratch holds one fp32 bin");
    static_assert(ONE_DIR || !TABLE, "the weight table is one direction's");
    static_assert(!RECORD || (NB == 1 && !BRICK && !STEP && !JVP && !KTRI), "RECORD: the plain forward march, one bin per thread");
    __shared__ __align__(16) TableRow table[TABLE ? kThreads / 32 : 1][32];
    __shared__ Fx96 ref[TABLE ? kThreads / 32 : 1][6];      // per warp: fraction of x_0 (cell word 0) and increment, per axis
    if (P.same_frac && (*P.same_frac != 0) != TABLE) return;           // the other instantiation marches this call
    const BrickGeom G = brick_geom(P.nx, P.ny, P.nz);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // A warp marches as a whole (its phases are warp votes): a lane without a ray of its own (padding slot, ragged
    // end) marches the ray of the warp's first live lane, DARK (exp(-tau) = 0: every deposit is an exact zero and is
    // never issued).  A warp with no live lane skips the march.
    RayId id;
    const bool live = ray_id(P, id);
    const unsigned live_mask = __ballot_sync(0xFFFFFFFFu, live);
    if (live_mask) {
        const int leader = __ffs(live_mask) - 1;
        const int lsrc = __shfl_sync(0xFFFFFFFFu, id.src, leader), lgroup = __shfl_sync(0xFFFFFFFFu, id.group, leader);
        const uint32_t lindex = __shfl_sync(0xFFFFFFFFu, id.index, leader);
        if (!live) { id.src = lsrc; id.group = lgroup; id.index = lindex; }

        PhasedLane<NB, ACC, JVP, KTRI> L;
        L.sg = sizeof(ACC) == 4 ? reinterpret_cast<ACC*>(P.scratch) : static_cast<ACC*>(P.acc);
        int negbits = 0;
        {
            double nh[3];
            fib_direction(id.index, uint32_t(P.n_rays), nh);
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const bool neg = nh[a] < 0.0;
                L.A[a].p = fx_from_double(source_coord(P, id.src, a), neg ? kFxComplement : kFxPlain);
                L.A[a].d = fx_from_double(__dmul_rn(P.ds, nh[a]), neg ? kFxNegate : kFxPlain);
                negbits |= neg ? (1 << a) : 0;
                if (TABLE && lane == 0) {
                    ref[warp][a] = Fx96{0, L.A[a].p.fh, L.A[a].p.fl};
                    ref[warp][3 + a] = L.A[a].d;
                }
                if (STEP) fx_advance(L.A[a].p, L.A[a].d, P.k0);      // x_k0 = x_0 + k0 ds n
            }
        }
        asm volatile("" : "+r"(negbits));        // opaque: keeps ptxas from re-deriving the signs with fp64 compares
        // One direction per warp, one bin: the signs are the same in every lane.  Passing them through a vote says so: they
        // live in uniform registers and what is derived from them runs on the uniform datapath (C2 11.84 -> 11.71 ms,
        // jittered C2 24.1 -> 22.7; with four bins per thread, C3, it makes no difference)
        if constexpr (ONE_DIR && NB == 1)
            negbits = (__any_sync(0xFFFFFFFFu, (negbits & 1) != 0) ? 1 : 0) | (__any_sync(0xFFFFFFFFu, (negbits & 2) != 0) ? 2 : 0) |
                      (__any_sync(0xFFFFFFFFu, (negbits & 4) != 0) ? 4 : 0);
#pragma unroll
        for (int s = 0; s < 8; ++s) L.S.zero_slot(s);
        L.S.restart(P, L.A, negbits, id.group * NB, P.j);
#pragma unroll
        for (int b = 0; b < NB; ++b) { L.I[b] = 0.0f; L.T[b] = live ? P.emis : 0.0f; }       // ds 4 pi/N_Omega rides on exp(-tau)
        if constexpr (JVP) {
#pragma unroll
            for (int b = 0; b < NB; ++b) { L.Id[b] = 0.0f; L.Td[b] = 0.0f; }
        }
        const size_t state_at = (size_t(id.src) * P.n_rays + id.index) * P.nb + size_t(id.group) * NB;
        if (STEP && live) {                  // the ray's (I, exp(-tau)) carried from the previous call
            const BinVec<NB> si = ld_bins<NB>(P.state_I + state_at), sT = ld_bins<NB>(P.state_T + state_at);
#pragma unroll
            for (int b = 0; b < NB; ++b) { L.I[b] = si.v[b]; L.T[b] = sT.v[b]; }
        }
        if constexpr (KTRI) {
#pragma unroll
            for (int b = 0; b < NB; ++b) L.att[b] = 1.0f;
        } else {
            phased_load_att<NB, JVP, !TABLE>(P, L, L.S.base + ((negbits & 1) ? L.A[0].dl : 0) + ((negbits & 2) ? L.A[1].dl : 0) +
                                          ((negbits & 4) ? L.A[2].dl : 0));
        }
        L.g = 0;
        L.rec_at = live ? (long long)blockIdx.x * kThreads + threadIdx.x : -1;
        L.left = (STEP && P.first_left) ? P.first_left : P.n_sub;
        L.roff = 0;
        L.woff = 0;
        if constexpr (BRICK)
            L.woff = (aidx<0>(P, L.A[0].p.c, negbits) * G.wy + aidx<1>(P, L.A[1].p.c, negbits) + ((negbits & 2) ? 0 : 1)) * G.sy +
                     (aidx<2>(P, L.A[2].p.c, negbits) + ((negbits & 4) ? 0 : 1)) * 4;
        __syncwarp();
        // shared-window address of this warp's table, kept in a register (opaque to the compiler, which would
        // otherwise rebuild it from the thread index every substep)
        uint32_t tbase = 0;
        if constexpr (TABLE) {
            tbase = uint32_t(__cvta_generic_to_shared(&table[warp][0]));
            asm volatile("" : "+r"(tbase));
        }
        // axes every ray of the warp has already left for good at x_0 (sources on or beyond a face)
        int act = 0;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const int lim = (a == 0 ? P.nx : (a == 1 ? P.ny : P.nz)) - 1;
            const bool gone = L.A[a].p.c >= ((negbits & (1 << a)) ? 0 : lim);
            if (!__all_sync(0xFFFFFFFFu, gone)) act |= 1 << a;
        }
        const int K = P.n_steps * P.n_sub - ((STEP && P.first_left) ? P.n_sub - P.first_left : 0);
        while (L.g < K) {
            if constexpr (TABLE) {
                if (L.roff == 0 && act != 0) {       // the table has run out: lane l writes the row of substep g + l
                    __syncwarp();
                    TableRow row;
                    row.pad[0] = row.pad[1] = 0;
#pragma unroll
                    for (int a = 0; a < 3; ++a) {
                        Fx96 p = ref[warp][a];
                        const Fx96 d = ref[warp][3 + a];
                        fx_advance(p, d, (STEP ? P.k0 : 0) + (long long)L.g + lane);
                        const uint32_t h = p.fh;
                        const int c = p.c;
                        fx_add(p, d);
                        const float t = __uint2float_rn(~h) * 2.3283064365386963e-10f;      // 2^-32
                        row.t[a][0] = (p.c != c) ? -t : t;
                        row.t[a][1] = __uint2float_rn(h) * 2.3283064365386963e-10f;
                    }
                    table[warp][lane] = row;
                    __syncwarp();
                }
            }
            switch (act) {
                case 7: act = phase<7, NB, TABLE, BRICK, STEP, JVP, KTRI, RECORD>(P, G, L, negbits, tbase); break;
                case 6: act = phase<6, NB, TABLE, BRICK, STEP, JVP, KTRI, RECORD>(P, G, L, negbits, tbase); break;
                case 5: act = phase<5, NB, TABLE, BRICK, STEP, JVP, KTRI, RECORD>(P, G, L, negbits, tbase); break;
                case 4: act = phase<4, NB, TABLE, BRICK, STEP, JVP, KTRI, RECORD>(P, G, L, negbits, tbase); break;
                case 3: act = phase<3, NB, TABLE, BRICK, STEP, JVP, KTRI, RECORD>(P, G, L, negbits, tbase); break;
                case 2: act = phase<2, NB, TABLE, BRICK, STEP, JVP, KTRI, RECORD>(P, G, L, negbits, tbase); break;
                case 1: act = phase<1, NB, TABLE, BRICK, STEP, JVP, KTRI, RECORD>(P, G, L, negbits, tbase); break;
                default: act = phase<0, NB, TABLE, BRICK, STEP, JVP, KTRI, RECORD>(P, G, L, negbits, tbase); break;
            }
            if (L.left == 0) {               // time-step boundary: the increments of this step are complete (rays continue, D7)
                if constexpr (RECORD) {
                    // nothing was deposited
                } else if constexpr (BRICK) {
                    brick_flush<-1, 7>(G, L, negbits);         // slots of inactive axes hold exact zeros: skipped by value
#pragma unroll
                    for (int s = 0; s < 8; ++s) L.S.zero_slot(s);
                    L.sg += G.step_stride;
                } else {
                    L.S.flush_all(L.sg, L.A);
                    L.sg += P.snap_stride;
                }
                L.left = P.n_sub;
            }
        }
        if (STEP && live) {
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                P.state_I[state_at + b] = L.I[b];
                P.state_T[state_at + b] = L.T[b];
            }
        }
    }
    if constexpr (RECORD || sizeof(ACC) == 8) return;
    // this block's turn at the drain: one slice of the scratch goes to the fp64 grid (rt_brick.cuh)
    const long long per = P.drain_units_per_block;
    if (per == 0) return;        // the scratch is the result grid itself: nothing to drain (rt_api.cu)
    const long long n_slices = (P.n_drain_units + per - 1) / per;
    const long long b0 = (blockIdx.x % n_slices) * per;
    if constexpr (BRICK)
        drain_bricks(P.scratch, static_cast<double*>(P.acc), G, P.nx, P.ny, P.nz, b0, min(b0 + per, P.n_drain_units), threadIdx.x,
                     kThreads);
    else
        drain_plain(P.scratch, static_cast<double*>(P.acc), b0, min(b0 + per, P.n_drain_units), threadIdx.x, kThreads);
}

}  // namespace rt
