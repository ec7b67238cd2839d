// rt_march_table.cuh — the sliding-stencil march for sources that share their cell fractions (sm_100a).
//
// With cell-centred sources (the paper places them at density-peak cells; BASELINE.json configs 2, 3)
// the 32 rays of a warp -- 32 sources, ONE direction -- have the SAME fractional position at every substep: they
// differ by whole cells.  Their trilinear weights, the fixed-point advance and the cell-crossing test are then the
// same numbers in every lane.  march_sliding_kernel computes them 32 times per substep; here the warp computes
// them once: every 32 substeps lane l evaluates substep g + l -- x_{g+l} = x_0 + (g + l) ds n in the same 96-bit
// arithmetic, its fraction words and which axes cross a cell plane -- into a 512-byte shared-memory table, and
// for the next 32 substeps every lane reads its row back (one 16-byte broadcast load; the L1/shared data pipe is
// the busiest unit of this kernel, so the row is as small as it can be).  Per lane remain: the clamping masks (an
// axis whose two indices clamp to one voxel takes the pair (1, 0)), the conversions and the 12 weight
// products, gather, eq. (2), deposit, and the slides.
// Every ray's arithmetic is bit for bit that of march_sliding_kernel; only the order of the reductions differs.
//
// The kernel runs only when `*P.same_frac` says that all sources of the call have equal fractions (decided on the
// device by same_fraction_kernel; otherwise it returns at once and march_sliding_kernel<..., COPIES>, launched
// right after with the complementary test, does the work).
//
// Registers: without the per-lane position and increment words the kernel fits 48 registers (4 bytes spilled), i.e.
// 10 blocks = 40 warps per SM against march_sliding_kernel's 8 blocks at 64 registers; that, not the saved
// instructions, is what it gains (C2: 17.2 ms at 8 blocks/SM -- the same as march_sliding_kernel -- 16.9 at 9, 16.8
// at 10, 21.0 at 12 with 76 bytes spilled).  Like march_sliding_kernel<..., COPIES> it spreads its reductions over
// the copies of the accumulation grid.
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

// number of slots in use below s (slots in use: those with no bit outside `bits`)
__host__ __device__ constexpr int slot_rank(int s, int bits) {
    int r = 0;
    for (int t = 0; t < s; ++t) r += ((t & ~bits) == 0) ? 1 : 0;
    return r;
}

// The state one lane carries through the march of march_table_kernel
struct TableLane {
    Stencil<1, double, false> S;
    TravelAxis A[3];         // only the cell word, dl and fmask are used
    float I, T, att;         // I scaled by 4 pi/N_Omega; T = exp(-tau) ds 4 pi/N_Omega; att = exp(-kappa ds) of the kappa cell
    float* sg;               // brick scratch of the current time step (rt_brick.cuh)
    int woff;                // float offset in it of the window the trailing slots start (lower index of y and z)
    int g;                   // substep index since x_0
    int left;                // substeps left in the current time step
    uint32_t roff;           // byte offset of the row of substep g in the warp's table
};

// array index of u-cell c of axis AX (c, or -c on a descending axis), clamped to the grid
template <int AX> __device__ __forceinline__ int aidx(const MarchParams& P, int c, int negbits) {
    const int lim = (AX == 0 ? P.nx : (AX == 1 ? P.ny : P.nz)) - 1;
    return min(max((negbits & (1 << AX)) ? -c : c, 0), lim);
}

// The pending sums of the lane's stencil as brick payloads (rt_brick.cuh).  Slots are [x][y][z] roles, 0 = trailing /
// 1 = leading in TRAVEL order; a brick is in ARRAY order, so on a descending axis the leading slot is the lower
// element.  The lower index of an axis is (trailing index - 1 on a descending axis), also when the axis is merged:
// the other element of the pair is then padding or a neighbour and carries the leading slot's exact zero.  Slots on
// the leading side of an inactive axis (ACT) do not exist: zero.
template <int ACT> struct BrickView {
    const Stencil<1, double, false>& S;
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
template <int AX, int ACT>
__device__ __forceinline__ void brick_flush(const BrickGeom& G, TableLane& L, int negbits) {
    const BrickView<ACT> V{L.S, (negbits & 2) != 0, (negbits & 4) != 0};
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

// PHASES.  ACT = set of ACTIVE axes (bit a).  An axis becomes inactive once EVERY ray of the warp has left the box
// through it for good -- travel-coordinate cell word beyond the far face; cell words only go up, so it stays merged
// (rt_march_sliding.cuh) for the rest of the march: its leading weight is 0 and its trailing weight 1 for every lane.
// The rays of a warp are parallel and their sources mostly neighbours, so they leave through the same faces at
// about the same time (C2: of 444 substeps a warp spends 148 with three active axes, 158 with two, 112 with one, 26
// with none).  table_phase<ACT> is the substep loop with the inactive axes compiled out: 2^n stencil slots (gather,
// deposit, weights), slides and crossing tests for the n active axes only -- the same sums, without the terms that
// are exactly zero.  It returns the next set of active axes (the warp-uniform vote after a cell crossing), or ACT
// when the last substep is done.
template <int ACT>
__device__ __forceinline__ int table_phase(const MarchParams& P, const BrickGeom& G, TableLane& L, int negbits,
                                           uint32_t tbase) {
    constexpr int kBits = ((ACT & 1) ? 4 : 0) | ((ACT & 2) ? 2 : 0) | ((ACT & 4) ? 1 : 0);      // slot index bits in use
    auto load_att = [&]() {
        int ko = L.S.base;
        if (ACT & 1) ko += (negbits & 1) ? L.A[0].dl : 0;
        if (ACT & 2) ko += (negbits & 2) ? L.A[1].dl : 0;
        if (ACT & 4) ko += (negbits & 4) ? L.A[2].dl : 0;
        L.att = ex2_approx(__ldg(P.kappa + ko) * P.att_scale);
    };
    int next = ACT;
    do {                                     // until the table runs out, the time step ends or an axis goes inactive
        float w[8];
        bool cross[3] = {false, false, false};
        if constexpr (ACT != 0) {
            float t[3] = {1.0f, 1.0f, 1.0f}, l[3] = {0.0f, 0.0f, 0.0f};
#pragma unroll
            for (int a = 0; a < 3; ++a)
                if (ACT & (1 << a)) {
                    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(t[a]), "=f"(l[a]) : "r"(tbase + L.roff + 8u * a));
                    cross[a] = __float_as_int(t[a]) < 0;
                    mask_pair(t[a], l[a], L.A[a].fmask);
                    t[a] = fabsf(t[a]);
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
        L.roff = (L.roff + 32u) & 1023u;
        float jv = 0.0f, ju = 0.0f;          // two partial sums over alternate slots: half the dependent-FMA chain length
        if constexpr (ACT == 0) {
            jv = L.S.jc[0].v[0];
        } else {
#pragma unroll
            for (int s = 0; s < 8; ++s)
                if ((s & ~kBits) == 0) {
                    const int r = slot_rank(s, kBits);           // position of s among the slots in use
                    const float jc = L.S.jc[s].v[0];
                    if (r & 1) ju = (r == 1) ? w[s] * jc : fmaf(w[s], jc, ju);
                    else jv = (r == 0) ? w[s] * jc : fmaf(w[s], jc, jv);
                }
        }
        L.I = fmaf(L.I, L.att, (jv + ju) * L.T);                           // eq. (2)
        L.T *= L.att;
#pragma unroll
        for (int s = 0; s < 8; ++s)
            if ((s & ~kBits) == 0) L.S.acc[s].v[0] = (ACT == 0) ? L.S.acc[s].v[0] + L.I : fmaf(w[s], L.I, L.S.acc[s].v[0]);

        if constexpr (ACT != 0) {
            if (cross[0] | cross[1] | cross[2]) {     // warp-uniform
#pragma unroll
                for (int a = 0; a < 3; ++a)
                    if ((ACT & (1 << a)) && cross[a]) {
                        L.A[a].p.c += 1;
                        if (a == 0) L.S.template axis_step_with<0, ACT>(P, L.A, negbits, P.j, [&]() { brick_flush<0, ACT>(G, L, negbits); });
                        if (a == 1) L.S.template axis_step_with<1, ACT>(P, L.A, negbits, P.j, [&]() { brick_flush<1, ACT>(G, L, negbits); });
                        if (a == 2) L.S.template axis_step_with<2, ACT>(P, L.A, negbits, P.j, [&]() { brick_flush<2, ACT>(G, L, negbits); });
                        // every ray of the warp beyond the far face of this axis: it stays merged from here on
                        const int lim = (a == 0 ? P.nx : (a == 1 ? P.ny : P.nz)) - 1;
                        const bool gone = L.A[a].p.c >= ((negbits & (1 << a)) ? 0 : lim);
                        if (__all_sync(0xFFFFFFFFu, gone)) next &= ~(1 << a);
                    }
                load_att();
            }
        }
        ++L.g;
        --L.left;
    } while (L.roff != 0 && L.left != 0 && next == ACT);
    return next;
}

#ifndef RT_TABLE_MINB
#define RT_TABLE_MINB 8
#endif
template <int MINB>
__global__ void __launch_bounds__(kThreads, MINB) march_table_kernel(const MarchParams P) {
    __shared__ __align__(16) TableRow table[kThreads / 32][32];
    __shared__ Fx96 ref[kThreads / 32][6];           // per warp: fraction of x_0 (cell word 0) and increment, per axis
    if (!*P.same_frac) return;
    const BrickGeom G = brick_geom(P.nx, P.ny, P.nz);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // warp -> direction slot, lane -> source rank (ray_id with map_src = 1, one bin)
    const uint32_t chunks = (uint32_t(P.n_slots) + 3u) / 4u;
    const uint32_t slot_ix = (blockIdx.x % chunks) * 4u + uint32_t(warp);
    const uint32_t rank0 = (blockIdx.x / chunks) * 32u;
    uint32_t index = kPad;
    if (slot_ix < uint32_t(P.n_slots) && rank0 < uint32_t(P.n_src)) index = P.ray_order ? P.ray_order[slot_ix] : slot_ix;
    if (index != kPad && index < uint32_t(P.n_rays)) {                 // warp-uniform: nothing in the march is divergent
        const bool live = rank0 + lane < uint32_t(P.n_src);            // a padding lane marches rank0's ray, dark
        const uint32_t rank = live ? rank0 + lane : rank0;
        const int src = int(P.src_order ? P.src_order[rank] : rank);

        TableLane L;
        L.sg = P.scratch;
        int negbits = 0;
        {
            double nh[3];
            fib_direction(index, uint32_t(P.n_rays), nh);
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const bool neg = nh[a] < 0.0;
                L.A[a].p = fx_from_double(source_coord(P, src, a), neg ? kFxComplement : kFxPlain);
                L.A[a].d = fx_from_double(__dmul_rn(P.ds, nh[a]), neg ? kFxNegate : kFxPlain);
                negbits |= neg ? (1 << a) : 0;
                if (lane == 0) {
                    ref[warp][a] = Fx96{0, L.A[a].p.fh, L.A[a].p.fl};
                    ref[warp][3 + a] = L.A[a].d;
                }
            }
        }
        asm volatile("" : "+r"(negbits));
#pragma unroll
        for (int s = 0; s < 8; ++s) L.S.zero_slot(s);
        L.S.restart(P, L.A, negbits, 0, P.j);
        L.I = 0.0f;
        L.T = live ? P.emis : 0.0f;          // the emission weight ds 4 pi/N_Omega rides on exp(-tau)
        L.att = ex2_approx(__ldg(P.kappa + L.S.base + ((negbits & 1) ? L.A[0].dl : 0) + ((negbits & 2) ? L.A[1].dl : 0) +
                                 ((negbits & 4) ? L.A[2].dl : 0)) * P.att_scale);
        L.g = 0;
        L.left = P.n_sub;
        L.roff = 0;
        L.woff = (aidx<0>(P, L.A[0].p.c, negbits) * G.wy + aidx<1>(P, L.A[1].p.c, negbits) + ((negbits & 2) ? 0 : 1)) * G.sy +
                 (aidx<2>(P, L.A[2].p.c, negbits) + ((negbits & 4) ? 0 : 1)) * 4;
        __syncwarp();

        // shared-window address of this warp's table, kept in a register (opaque to the compiler, which would
        // otherwise rebuild it from the thread index every substep)
        uint32_t tbase = uint32_t(__cvta_generic_to_shared(&table[warp][0]));
        asm volatile("" : "+r"(tbase));

        // axes every ray of the warp has already left for good at x_0 (sources on or beyond a face)
        int act = 0;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const int lim = (a == 0 ? P.nx : (a == 1 ? P.ny : P.nz)) - 1;
            const bool gone = L.A[a].p.c >= ((negbits & (1 << a)) ? 0 : lim);
            if (!__all_sync(0xFFFFFFFFu, gone)) act |= 1 << a;
        }
        const int K = P.n_steps * P.n_sub;
        while (L.g < K) {
            if (L.roff == 0 && act != 0) {   // the table has run out: lane l writes the row of substep g + l
                __syncwarp();
                TableRow row;
                row.pad[0] = row.pad[1] = 0;
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    Fx96 p = ref[warp][a];
                    const Fx96 d = ref[warp][3 + a];
                    fx_advance(p, d, (long long)L.g + lane);
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
            switch (act) {
                case 7: act = table_phase<7>(P, G, L, negbits, tbase); break;
                case 6: act = table_phase<6>(P, G, L, negbits, tbase); break;
                case 5: act = table_phase<5>(P, G, L, negbits, tbase); break;
                case 4: act = table_phase<4>(P, G, L, negbits, tbase); break;
                case 3: act = table_phase<3>(P, G, L, negbits, tbase); break;
                case 2: act = table_phase<2>(P, G, L, negbits, tbase); break;
                case 1: act = table_phase<1>(P, G, L, negbits, tbase); break;
                default: act = table_phase<0>(P, G, L, negbits, tbase); break;
            }
            if (L.left == 0) {               // time-step boundary: the increments of this step are complete (rays continue, D7)
                brick_flush<-1, 7>(G, L, negbits);               // slots of inactive axes hold exact zeros: skipped by value
#pragma unroll
                for (int s = 0; s < 8; ++s) L.S.zero_slot(s);
                L.sg += G.step_stride;
                L.left = P.n_sub;
            }
        }
    }
    // this block's turn at the drain: one slice of the scratch goes to the fp64 grid (rt_brick.cuh)
    const long long per = P.drain_bricks_per_block;
    const long long n_slices = (P.n_bricks + per - 1) / per;
    const long long b0 = (blockIdx.x % n_slices) * per;
    drain_bricks(P.scratch, static_cast<double*>(P.acc), G, P.nx, P.ny, P.nz, b0, min(b0 + per, P.n_bricks), threadIdx.x,
                 kThreads);
}

}  // namespace rt
