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

struct TableRow {            // substep g of a direction: 32 bytes, two 16-byte shared-memory loads per substep
    float tx, lx, ty, ly;    // trailing / leading weight of x_g per axis, unscaled: float(~h), float(h) of the top 32
    float tz, lz;            // fraction bits h (travel coordinates, rt_march_sliding.cuh); the z pair carries 2^-96
    int cross;               // bit a: the cell word of axis a goes up between x_g and x_{g+1}
    int pad;
};

// (t, l) of an axis with the clamping mask of the lane applied: m = ~0 leaves the pair, m = 0 -- both
// indices of the axis clamp to one voxel -- makes it exactly (one, 0), `one` being float(~0u) = 2^32 (times 2^-96 on z).
// The same values as masking the fraction word before the conversions, bit for bit.
__device__ __forceinline__ void mask_pair(float& t, float& l, uint32_t m, uint32_t one_bits) {
    t = __uint_as_float((__float_as_uint(t) & m) | (one_bits & ~m));
    l = __uint_as_float(__float_as_uint(l) & m);
}

template <int MINB>
__global__ void __launch_bounds__(kThreads, MINB) march_table_kernel(const MarchParams P) {
    __shared__ __align__(16) TableRow table[kThreads / 32][32];
    __shared__ Fx96 ref[kThreads / 32][6];           // per warp: fraction of x_0 (cell word 0) and increment, per axis
    if (!*P.same_frac) return;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // warp -> direction slot, lane -> source rank (ray_id with map_src = 1, one bin)
    const uint32_t chunks = (uint32_t(P.n_slots) + 3u) / 4u;
    const uint32_t slot_ix = (blockIdx.x % chunks) * 4u + uint32_t(warp);
    const uint32_t rank0 = (blockIdx.x / chunks) * 32u;
    if (slot_ix >= uint32_t(P.n_slots) || rank0 >= uint32_t(P.n_src)) return;
    const uint32_t index = P.ray_order ? P.ray_order[slot_ix] : slot_ix;
    if (index == kPad || index >= uint32_t(P.n_rays)) return;          // warp-uniform: nothing below is divergent
    const bool live = rank0 + lane < uint32_t(P.n_src);                // a padding lane marches rank0's ray, dark
    const uint32_t rank = live ? rank0 + lane : rank0;
    const int src = int(P.src_order ? P.src_order[rank] : rank);
    double* og = static_cast<double*>(P.acc) + (blockIdx.x % unsigned(P.acc_copies)) * P.acc_copy_stride;

    TravelAxis A[3];                         // only the cell word, dl and fmask are used here
    int negbits = 0;
    {
        double nh[3];
        fib_direction(index, uint32_t(P.n_rays), nh);
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const bool neg = nh[a] < 0.0;
            A[a].p = fx_from_double(source_coord(P, src, a), neg ? kFxComplement : kFxPlain);
            A[a].d = fx_from_double(__dmul_rn(P.ds, nh[a]), neg ? kFxNegate : kFxPlain);
            negbits |= neg ? (1 << a) : 0;
            if (lane == 0) {
                ref[warp][a] = Fx96{0, A[a].p.fh, A[a].p.fl};
                ref[warp][3 + a] = A[a].d;
            }
        }
    }
    asm volatile("" : "+r"(negbits));
    Stencil<1, double, false> S;
#pragma unroll
    for (int s = 0; s < 8; ++s) S.zero_slot(s);
    S.restart(P, A, negbits, 0, P.j);
    float I = 0.0f, T = live ? P.emis : 0.0f, att;   // T = exp(-tau) ds 4 pi/N_Omega: the emission weight rides on it
    auto load_att = [&]() {
        const int ko = S.base + ((negbits & 1) ? A[0].dl : 0) + ((negbits & 2) ? A[1].dl : 0) + ((negbits & 4) ? A[2].dl : 0);
        att = ex2_approx(__ldg(P.kappa + ko) * P.att_scale);
    };
    load_att();
    __syncwarp();

    // shared-window address of this warp's table, kept in a register (opaque to the compiler, which would
    // otherwise rebuild it from the thread index every substep), and the byte offset of the current row
    uint32_t tbase = uint32_t(__cvta_generic_to_shared(&table[warp][0]));
    asm volatile("" : "+r"(tbase));
    uint32_t roff = 0;

    int g = 0;                               // substep index since x_0
    for (int m = 0; m < P.n_steps; ++m) {
        for (int k = 0; k < P.n_sub; ++k, ++g) {
            if (roff == 0) {                 // lane l writes the row of substep g + l
                __syncwarp();
                TableRow row;
                row.cross = 0;
                row.pad = 0;
                uint32_t h[3];
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    Fx96 p = ref[warp][a];
                    const Fx96 d = ref[warp][3 + a];
                    fx_advance(p, d, (long long)g + lane);
                    h[a] = p.fh;
                    const int c = p.c;
                    fx_add(p, d);
                    row.cross |= (p.c != c) ? (1 << a) : 0;
                }
                row.tx = __uint2float_rn(~h[0]); row.lx = __uint2float_rn(h[0]);
                row.ty = __uint2float_rn(~h[1]); row.ly = __uint2float_rn(h[1]);
                row.tz = __uint2float_rn(~h[2]) * 1.2621774483536189e-29f;      // 2^-96
                row.lz = __uint2float_rn(h[2]) * 1.2621774483536189e-29f;
                table[warp][lane] = row;
                __syncwarp();
            }
            float4 rxy, rz;
            asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];"
                         : "=f"(rxy.x), "=f"(rxy.y), "=f"(rxy.z), "=f"(rxy.w) : "r"(tbase + roff));
            asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4+16];"
                         : "=f"(rz.x), "=f"(rz.y), "=f"(rz.z), "=f"(rz.w) : "r"(tbase + roff));
            roff = (roff + 32u) & 1023u;
            // from here on the substep is march_sliding_kernel's: the lane's clamping masks, unscaled weights, 2^-96 on z
            float tx = rxy.x, lx = rxy.y, ty = rxy.z, ly = rxy.w, tz = rz.x, lz = rz.y;
            mask_pair(tx, lx, A[0].fmask, 0x4F800000u);          // 2^32
            mask_pair(ty, ly, A[1].fmask, 0x4F800000u);
            mask_pair(tz, lz, A[2].fmask, 0x1F800000u);          // 2^-64 = 2^32 2^-96
            const int cross = __float_as_int(rz.z);
            const float wz[2] = {tz, lz};
            const float wxy[4] = {tx * ty, tx * ly, lx * ty, lx * ly};
            float w[8];
#pragma unroll
            for (int s = 0; s < 8; ++s) w[s] = wxy[s >> 1] * wz[s & 1];
            float jv = w[0] * S.jc[0].v[0], ju = w[1] * S.jc[1].v[0];
#pragma unroll
            for (int s = 2; s < 8; s += 2) {
                jv = fmaf(w[s], S.jc[s].v[0], jv);
                ju = fmaf(w[s + 1], S.jc[s + 1].v[0], ju);
            }
            I = fmaf(I, att, (jv + ju) * T);                           // eq. (2)
            T *= att;
#pragma unroll
            for (int s = 0; s < 8; ++s) S.acc[s].v[0] = fmaf(w[s], I, S.acc[s].v[0]);

            if (cross) {                     // warp-uniform
                if (cross & 1) { A[0].p.c += 1; S.template axis_step<0>(P, A, negbits, og, P.j); }
                if (cross & 2) { A[1].p.c += 1; S.template axis_step<1>(P, A, negbits, og, P.j); }
                if (cross & 4) { A[2].p.c += 1; S.template axis_step<2>(P, A, negbits, og, P.j); }
                load_att();
            }
        }
        S.flush_all(og, A);    // time-step boundary (rays continue, D7)
        og += P.snap_stride;
    }
}

}  // namespace rt
