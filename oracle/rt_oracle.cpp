// rt_oracle.cpp — fp64 CPU ORACLE for the Ray-trax ray march.  TEST INFRASTRUCTURE ONLY.
//
// This file is the plain, slow, obviously-correct restatement of what the hot path computes, written
// from the paper (/root/reference/PAPER.md, cited below as P:<line>) and from nothing else.  It shares
// no code, header or table with the CUDA path under paper_2511_09389_b200/csrc/, and neither side
// includes or links the other.  What the two sides do share is a READING, D1/D3: positions live
// on a 2^-64 cell grid and the azimuth is reduced with the golden turn as a 128-bit fixed-point fraction, so
// the same mathematical constants ((3 - sqrt 5)/2 * 2^128, 2^-64) appear on both sides, each written out
// separately; floor(x_k) on tie rays then agrees by construction of the reading, not by a shared routine.
// The guards that are independent of both are the pins: the lattice against 50-digit arithmetic (P0) and the
// positions against exact rationals (fractions.Fraction, D3) in tests/test_oracle_pins.py.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs may build,
// load or call it.  The product path never routes through it.
//
// What it computes (eq. (2) at P:23; readings D1..D16 are listed in DESIGN.md §4):
//
//   N_s   = substeps(step_size, c, dt)                                   P:25   (reading D6)
//   acc[nx][ny][nz][B] = 0
//   for m in 0 .. n_steps-1:                                             P:56, P:35 (reading D7: rays continue)
//     for every source s and every Fibonacci direction i (any order; state I[b], tau[b] kept per (s,i)):
//       nhat = fib(i, N_Omega)                                           P:27   (reading D1)
//       for k in m*N_s .. (m+1)*N_s - 1:
//         p   = x0[s] + k * (ds * nhat)   on the 2^-64 cell grid         P:23   (x_{k+1} = x_k + nhat ds, closed form, D3)
//         i0  = floor(p) per axis;  f = p - i0 in [0,1)
//         lo  = clamp(i0, 0, N-1);  hi = clamp(i0+1, 0, N-1)             P:29   "Indexing is clamped" (D5)
//         for every bin b:                                               P:39   bins are a batch axis
//           kap = kappa[lo0][lo1][lo2][b]                                P:29   nearest-neighbour at the cell of x_k (D4)
//           jv  = sum over the 8 corners of w_c * j[corner_c][b]         P:29   trilinear read of j at x_k
//           I[b]   = I[b]*exp(-kap*ds) + jv*exp(-tau[b])*ds              P:23   eq. (2), uses tau_k
//           tau[b] = tau[b] + kap*ds
//           acc[corner_c][b] += w_c * I[b]   for the same 8 corners      P:29   deposit I_{k+1}, same weights (D2)
//     out[m] = (4 pi / N_Omega) * acc                                    P:27   (cumulative snapshot, D7/D8)
//
// Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): closed form in a uniform medium, deposit-mass
// conservation, N_Omega invariance, the analytic point source of P:45 (eq. 3), the light-front horizon,
// hand-unrolled traces on 4^3 grids, the prefix property, the optically thin limit, linearity /
// additivity / bin independence, trilinear consistency, and the direction lattice against 50-digit
// arithmetic.  Reading D4 (floor vs round for "nearest neighbour") and the exact lattice D1 are pinned
// only by those hand traces and by DESIGN.md's decision: the paper itself does not fix them.
//
// All arithmetic is double, except: long double to reduce the golden-angle phase accurately, and the position
// x_k, which is evaluated EXACTLY on a 2^-64 cell grid in 128-bit integers (reading D3) so that floor(x_k) is the
// same decision for every implementation of that reading.  No SIMD, no
// blocking, no reordering beyond "rays are independent": rays are split over threads, each thread
// owns a private grid, and the private grids are added in thread order, so a run is bit-reproducible for a
// given thread count.
#include <algorithm>
#include <cmath>
#include <cstddef>
#include <cstdint>
#include <thread>
#include <vector>

namespace {

constexpr long double kPiL = 3.14159265358979323846264338327950288L;

struct Medium {
    const float* j;
    const float* kappa;
    long nx, ny, nz, nb;
    bool ktri = false;   // reading D18: kappa read by trilinear interpolation (the weights of j) instead of nearest neighbour
    size_t cell(long a, long b, long c) const { return ((size_t(a) * ny + b) * nz + c) * nb; }
};

// P:25 / reading D6: N_s = ceil(c dt / ds); a ratio within 1e-6 (relative) of an integer is that integer
// (step_size, c, dt arrive as fp32, so e.g. 0.3f/0.1f = 3.00000007 must give 3, not 4).
long substeps(double ds, double c, double dt) {
    double r = c * dt / ds;
    double rr = std::round(r);
    if (rr >= 1.0 && std::fabs(r - rr) <= 1e-6 * r) return long(rr);
    return long(std::ceil(r));
}

// P:27 / reading D1: golden-angle lattice, i = 0..n-1, z_i = 1 - (2i+1)/n = (n-2i-1)/n, phi_i = i * pi * (3 - sqrt 5).
// z and the radius sqrt((1-z)(1+z)) are formed from exact integers with correctly rounded IEEE double operations
// only (one division for z; two divisions, one product, one square root for the radius), so that any
// implementation stating the same operations gets the same bits: z decides floor() ties of rational positions
// (reading D3).  The azimuth is reduced in long double with a two-term golden-angle constant.
void fib_direction(long i, long n, double nhat[3]) {
    const double dn = double(n), di = double(i);
    volatile double one_minus_z = (2.0 * di + 1.0) / dn;
    volatile double one_plus_z = (2.0 * double(n - i) - 1.0) / dn;
    volatile double prod = one_minus_z * one_plus_z;
    const double r = std::sqrt(prod);
    // phi / (2 pi) mod 1 = frac(i g), g = (3 - sqrt 5)/2 = 0x0.61C8864680B583EA0C633F9FA31237CB... split into two
    // exactly representable long doubles; the product i*g_hi is taken with its exact residual (fmal), so the
    // reduced turn is good to ~1e-19 for every i < 2^30 (a plain long double product loses i * 2^-64 turn).
    const long double g_hi = 0x61C8864680B583EAp-64L, g_lo = 0x0C633F9FA31237CBp-128L, li = (long double)i;
    const long double p = li * g_hi;
    const long double resid = fmal(li, g_hi, -p);
    long double turn = (p - floorl(p)) + (resid + li * g_lo);
    long double phi = 2.0L * kPiL * turn;
    volatile double c = double(cosl(phi)), s = double(sinl(phi));
    nhat[0] = r * c;
    nhat[1] = r * s;
    nhat[2] = (dn - 2.0 * di - 1.0) / dn;
}

// Reading D3: positions live on the 2^-64 cell grid.  fx(v) = floor(v * 2^64) EXACTLY (the double's significand is
// shifted, nothing is rounded), and x_k := (fx(x_0) + k * fx(ds * nhat)) / 2^64 in exact integer arithmetic, so
// floor(x_k) -- the one discontinuous decision of the method (nearest-neighbour kappa) -- does not depend on
// floating-point rounding order.  |x_k - (x_0 + k ds nhat)| < (k+1) 2^-64 cell.
typedef __int128 fx_t;

fx_t fx(double v) {
    if (v == 0.0) return 0;
    int e;
    const double m = std::frexp(v, &e);                   // v = m 2^e, 0.5 <= |m| < 1
    const long long M = (long long)std::ldexp(m, 53);     // exact 53-bit signed integer: v = M 2^(e-53)
    const int sh = e + 11;                                // v 2^64 = M 2^sh
    if (sh >= 0) return fx_t(M) << sh;                    // |v| < 2^30 in every caller: no overflow
    if (sh > -64) return fx_t(M >> (-sh));                // arithmetic shift of a negative value = floor
    return M < 0 ? -1 : 0;
}

inline long clampl(long v, long lo, long hi) { return v < lo ? lo : (v > hi ? hi : v); }

// Substeps k_begin .. k_end-1 of one ray, eq. (2) + deposit.  I/tau: per-bin state (in/out).
// trace_* (optional, may be null): per-substep records for the pin tests.
void march_ray(const Medium& M, const double x0[3], const double nhat[3], double ds, long k_begin, long k_end,
               double* I, double* tau, double* acc, double* trace_I, double* trace_tau, double* trace_pos) {
    const long N[3] = {M.nx, M.ny, M.nz};
    fx_t X0[3], D[3];
    for (int a = 0; a < 3; ++a) {
        X0[a] = fx(x0[a]);
        volatile double step = ds * nhat[a];              // one rounding, no contraction
        D[a] = fx(step);
    }
    for (long k = k_begin; k < k_end; ++k) {
        long lo[3], hi[3];
        double f[3];
        for (int a = 0; a < 3; ++a) {
            const fx_t X = X0[a] + fx_t(k) * D[a];        // x_k on the 2^-64 grid (reading D3)
            const long i0 = long((long long)(X >> 64));   // floor(x_k)
            const unsigned long long frac = (unsigned long long)X;
            f[a] = double(frac) * 5.42101086242752217e-20;   // (x_k - floor x_k), frac * 2^-64
            lo[a] = clampl(i0, 0, N[a] - 1);
            hi[a] = clampl(i0 + 1, 0, N[a] - 1);
            if (trace_pos) trace_pos[(k - k_begin) * 3 + a] = double(i0) + f[a];
        }
        size_t corner[8];
        double w[8];
        for (int c = 0; c < 8; ++c) {
            int dx = (c >> 2) & 1, dy = (c >> 1) & 1, dz = c & 1;
            corner[c] = M.cell(dx ? hi[0] : lo[0], dy ? hi[1] : lo[1], dz ? hi[2] : lo[2]);
            w[c] = (dx ? f[0] : 1.0 - f[0]) * (dy ? f[1] : 1.0 - f[1]) * (dz ? f[2] : 1.0 - f[2]);
        }
        const size_t base = M.cell(lo[0], lo[1], lo[2]);
        for (long b = 0; b < M.nb; ++b) {
            double kap = double(M.kappa[base + b]);                 // P:29 nearest neighbour at the cell of x_k (D4)
            if (M.ktri) {                                            // D18 variant: the same trilinear weights as j
                kap = 0.0;
                for (int c = 0; c < 8; ++c) kap += w[c] * double(M.kappa[corner[c] + b]);
            }
            double jv = 0.0;
            for (int c = 0; c < 8; ++c) jv += w[c] * double(M.j[corner[c] + b]);
            I[b] = I[b] * std::exp(-kap * ds) + jv * std::exp(-tau[b]) * ds;
            tau[b] = tau[b] + kap * ds;
            for (int c = 0; c < 8; ++c) acc[corner[c] + b] += w[c] * I[b];
            if (trace_I) trace_I[(k - k_begin) * M.nb + b] = I[b];
            if (trace_tau) trace_tau[(k - k_begin) * M.nb + b] = tau[b];
        }
    }
}

bool bad(double v) { return !(std::isfinite(v) && v > 0.0); }

}  // namespace

extern "C" {

// N_s as the oracle computes it (D6).  Returns -1 on invalid arguments.
long rt_oracle_substeps(float step_size, float c, float dt) {
    if (bad(step_size) || bad(c) || bad(dt)) return -1;
    return substeps(double(step_size), double(c), double(dt));
}

// Direction i of an n-point lattice (D1) -> nhat[3] (array axes 0,1,2).
int rt_oracle_direction(long i, long n, double* nhat) {
    if (n < 1 || i < 0 || i >= n || !nhat) return -1;
    fib_direction(i, n, nhat);
    return 0;
}

// One ray, n_sub substeps from k = 0 (I_0 = tau_0 = 0, D11).  Records I_{k+1}, tau_{k+1} and x_k for every
// substep and adds the UNNORMALISED deposits into acc (double [nx][ny][nz][B], caller-zeroed; may be null).
int rt_oracle_trace_ray_k(const float* j, const float* kappa, int nx, int ny, int nz, int n_bins,
                          const float* source_pos, long ray_index, long n_rays, float step_size, long n_sub,
                          double* trace_I, double* trace_tau, double* trace_pos, double* acc, int kappa_trilinear);

int rt_oracle_trace_ray(const float* j, const float* kappa, int nx, int ny, int nz, int n_bins,
                        const float* source_pos, long ray_index, long n_rays, float step_size, long n_sub,
                        double* trace_I, double* trace_tau, double* trace_pos, double* acc) {
    return rt_oracle_trace_ray_k(j, kappa, nx, ny, nz, n_bins, source_pos, ray_index, n_rays, step_size, n_sub,
                                 trace_I, trace_tau, trace_pos, acc, 0);
}

// The same with the kappa reading chosen: 0 = nearest neighbour (the paper), 1 = trilinear (D18).
int rt_oracle_trace_ray_k(const float* j, const float* kappa, int nx, int ny, int nz, int n_bins,
                          const float* source_pos, long ray_index, long n_rays, float step_size, long n_sub,
                          double* trace_I, double* trace_tau, double* trace_pos, double* acc, int kappa_trilinear) {
    if (!j || !kappa || !source_pos || nx < 1 || ny < 1 || nz < 1 || n_bins < 1 || n_sub < 0 || bad(step_size))
        return -1;
    Medium M{j, kappa, nx, ny, nz, n_bins, kappa_trilinear != 0};
    double nhat[3];
    if (rt_oracle_direction(ray_index, n_rays, nhat)) return -1;
    double x0[3] = {double(source_pos[0]), double(source_pos[1]), double(source_pos[2])};
    std::vector<double> I(n_bins, 0.0), tau(n_bins, 0.0), scratch;
    if (!acc) { scratch.assign(size_t(nx) * ny * nz * n_bins, 0.0); acc = scratch.data(); }
    march_ray(M, x0, nhat, double(step_size), 0, n_sub, I.data(), tau.data(), acc, trace_I, trace_tau, trace_pos);
    return 0;
}

// The multi-source march.  Host pointers.  out: double [n_steps][nx][ny][nz][n_bins],
// overwritten; snapshot m is cumulative (D7) and scaled once by 4 pi / N_Omega (D8).
// n_threads < 1 means 1.  Returns 0, or -1 on invalid arguments.
int rt_march_oracle_k(const float* j, const float* kappa, int nx, int ny, int nz, const float* sources, int n_src,
                      int n_rays, int n_bins, float step_size, float c, float dt, int n_steps, double* out,
                      int n_threads, int kappa_trilinear);

int rt_march_oracle(const float* j, const float* kappa, int nx, int ny, int nz, const float* sources, int n_src,
                    int n_rays, int n_bins, float step_size, float c, float dt, int n_steps, double* out,
                    int n_threads) {
    return rt_march_oracle_k(j, kappa, nx, ny, nz, sources, n_src, n_rays, n_bins, step_size, c, dt, n_steps, out,
                             n_threads, 0);
}

// The same with the kappa reading chosen: 0 = nearest neighbour (the paper), 1 = trilinear (D18).
int rt_march_oracle_k(const float* j, const float* kappa, int nx, int ny, int nz, const float* sources, int n_src,
                      int n_rays, int n_bins, float step_size, float c, float dt, int n_steps, double* out,
                      int n_threads, int kappa_trilinear) {
    if (!j || !kappa || !sources || !out) return -1;
    if (nx < 1 || ny < 1 || nz < 1 || n_src < 1 || n_rays < 1 || n_bins < 1 || n_steps < 1) return -1;
    if (bad(step_size) || bad(c) || bad(dt)) return -1;
    const long Ns = substeps(double(step_size), double(c), double(dt));
    const double ds = double(step_size);
    const Medium M{j, kappa, nx, ny, nz, n_bins, kappa_trilinear != 0};
    const size_t grid = size_t(nx) * ny * nz * n_bins;
    const long total_rays = long(n_src) * n_rays;
    long T = std::max(1, n_threads);
    T = std::min<long>(T, total_rays);

    std::vector<std::vector<double>> acc(T);                           // one private cumulative grid per thread
    std::vector<double> state(size_t(total_rays) * n_bins * 2, 0.0);   // (I[b], tau[b]) per ray; I_0 = tau_0 = 0
    for (auto& a : acc) a.assign(grid, 0.0);
    const double scale = double(4.0L * kPiL / (long double)n_rays);

    for (long m = 0; m < n_steps; ++m) {
        auto work = [&](long t) {
            long r0 = total_rays * t / T, r1 = total_rays * (t + 1) / T;   // contiguous chunk of (s, i) pairs
            for (long r = r0; r < r1; ++r) {
                long s = r / n_rays, i = r % n_rays;
                double nhat[3];
                fib_direction(i, n_rays, nhat);
                double x0[3] = {double(sources[3 * s]), double(sources[3 * s + 1]), double(sources[3 * s + 2])};
                double* I = &state[size_t(r) * n_bins * 2];
                march_ray(M, x0, nhat, ds, m * Ns, (m + 1) * Ns, I, I + n_bins, acc[t].data(), nullptr, nullptr,
                          nullptr);
            }
        };
        std::vector<std::thread> pool;
        for (long t = 1; t < T; ++t) pool.emplace_back(work, t);
        work(0);
        for (auto& th : pool) th.join();

        double* snap = out + size_t(m) * grid;
        auto reduce = [&](long t) {                                    // fixed order over the private grids
            size_t v0 = grid * size_t(t) / T, v1 = grid * size_t(t + 1) / T;
            for (size_t v = v0; v < v1; ++v) {
                double sum = 0.0;
                for (long u = 0; u < T; ++u) sum += acc[u][v];
                snap[v] = scale * sum;
            }
        };
        pool.clear();
        for (long t = 1; t < T; ++t) pool.emplace_back(reduce, t);
        reduce(0);
        for (auto& th : pool) th.join();
    }
    return 0;
}

// One time step with EXPLICIT ray state ("for strict time integration we fix dt and iterate"; P:58 RT substeps
// between hydro updates; reading D17): substeps k_begin .. k_begin + N_s - 1 of every ray, in the medium
// (j, kappa) passed to THIS call -- the caller may change it between calls.  Positions continue the same straight
// line, x_k = x_0 + k ds nhat; (I, tau) carry over in `state`.
//   state: double [n_src][n_rays][2][n_bins] = I[b] then tau[b] per ray; all zeros for a fresh start (D11); updated.
//   inc:   double [nx][ny][nz][n_bins], OVERWRITTEN with (4 pi / N_Omega) * the deposits of this step alone.
// With an unchanged medium the increments of successive calls add up to the cumulative snapshots of rt_march_oracle.
int rt_oracle_step(const float* j, const float* kappa, int nx, int ny, int nz, const float* sources, int n_src,
                   int n_rays, int n_bins, float step_size, float c, float dt, long k_begin, double* state,
                   double* inc, int n_threads) {
    if (!j || !kappa || !sources || !state || !inc) return -1;
    if (nx < 1 || ny < 1 || nz < 1 || n_src < 1 || n_rays < 1 || n_bins < 1 || k_begin < 0) return -1;
    if (bad(step_size) || bad(c) || bad(dt)) return -1;
    const long Ns = substeps(double(step_size), double(c), double(dt));
    const double ds = double(step_size);
    const Medium M{j, kappa, nx, ny, nz, n_bins};
    const size_t grid = size_t(nx) * ny * nz * n_bins;
    const long total_rays = long(n_src) * n_rays;
    long T = std::min<long>(std::max(1, n_threads), total_rays);
    std::vector<std::vector<double>> acc(T);
    for (auto& a : acc) a.assign(grid, 0.0);
    auto work = [&](long t) {
        long r0 = total_rays * t / T, r1 = total_rays * (t + 1) / T;
        for (long r = r0; r < r1; ++r) {
            long s = r / n_rays, i = r % n_rays;
            double nhat[3];
            fib_direction(i, n_rays, nhat);
            double x0[3] = {double(sources[3 * s]), double(sources[3 * s + 1]), double(sources[3 * s + 2])};
            double* I = state + size_t(r) * n_bins * 2;
            march_ray(M, x0, nhat, ds, k_begin, k_begin + Ns, I, I + n_bins, acc[t].data(), nullptr, nullptr, nullptr);
        }
    };
    std::vector<std::thread> pool;
    for (long t = 1; t < T; ++t) pool.emplace_back(work, t);
    work(0);
    for (auto& th : pool) th.join();
    const double scale = double(4.0L * kPiL / (long double)n_rays);
    for (size_t v = 0; v < grid; ++v) {
        double sum = 0.0;
        for (long u = 0; u < T; ++u) sum += acc[u][v];
        inc[v] = scale * sum;
    }
    return 0;
}

// ADJOINT of the march with respect to j ("its Jacobians with respect to (j, kappa) are well defined";
// DESIGN.md reading D19).  For fixed kappa the field is linear in j, out[m] = A_m j.  Given gbar[m] = dL/d out[m]
// this returns grad_j = sum_m A_m^T gbar[m], i.e. dL/dj.  Derived from eq. (2) and the deposit rule:
//   I_{k+1} = a_k I_k + T_k ds (w_k . j),  a_k = exp(-kappa_k ds),  T_k = exp(-tau_k);   out[m] += s w_k I_{k+1}
//   for every substep k of time steps 0..m, s = 4 pi / N_Omega.  Hence L = sum_k G_k I_{k+1} with
//   G_k = s w_k . (sum_{m >= step(k)} gbar[m]),   lambda_{k+1} := dL/dI_{k+1} = G_k + a_{k+1} lambda_{k+2} (lambda_{K+1} = 0),
//   grad_j[corner_c] += lambda_{k+1} T_k ds w_k[c].
// Written as it reads: a forward sweep that records (corners, weights, a_k, T_k) of every substep of a ray, then the
// backward recurrence.  gbar: double [n_steps][nx][ny][nz][B]; grad_j: double [nx][ny][nz][B], overwritten.
int rt_adjoint_j_oracle(const double* gbar, const float* kappa, int nx, int ny, int nz, const float* sources, int n_src,
                        int n_rays, int n_bins, float step_size, float c, float dt, int n_steps, double* grad_j,
                        int n_threads) {
    if (!gbar || !kappa || !sources || !grad_j) return -1;
    if (nx < 1 || ny < 1 || nz < 1 || n_src < 1 || n_rays < 1 || n_bins < 1 || n_steps < 1) return -1;
    if (bad(step_size) || bad(c) || bad(dt)) return -1;
    const long Ns = substeps(double(step_size), double(c), double(dt)), K = Ns * n_steps;
    const double ds = double(step_size);
    const long N[3] = {nx, ny, nz};
    const Medium M{nullptr, kappa, nx, ny, nz, n_bins};
    const size_t grid = size_t(nx) * ny * nz * n_bins;
    const double scale = double(4.0L * kPiL / (long double)n_rays);
    std::vector<double> gsuf(gbar, gbar + grid * size_t(n_steps));          // gsuf[m] = sum_{m' >= m} gbar[m']
    for (long m = n_steps - 2; m >= 0; --m)
        for (size_t v = 0; v < grid; ++v) gsuf[size_t(m) * grid + v] += gsuf[size_t(m + 1) * grid + v];
    const long total_rays = long(n_src) * n_rays;
    const long T = std::min<long>(std::max(1, n_threads), total_rays);
    std::vector<std::vector<double>> acc(T);
    for (auto& a : acc) a.assign(grid, 0.0);
    auto work = [&](long t) {
        std::vector<size_t> corner(size_t(K) * 8);
        std::vector<double> w(size_t(K) * 8), att(size_t(K) * n_bins), tr(size_t(K) * n_bins);
        for (long r = total_rays * t / T; r < total_rays * (t + 1) / T; ++r) {
            const long s = r / n_rays, i = r % n_rays;
            double nhat[3];
            fib_direction(i, n_rays, nhat);
            fx_t X0[3], D[3];
            for (int a = 0; a < 3; ++a) {
                X0[a] = fx(double(sources[3 * s + a]));
                volatile double step = ds * nhat[a];
                D[a] = fx(step);
            }
            std::vector<double> tau(n_bins, 0.0);
            for (long k = 0; k < K; ++k) {                                  // forward sweep: geometry, a_k, T_k
                long lo[3], hi[3];
                double f[3];
                for (int a = 0; a < 3; ++a) {
                    const fx_t X = X0[a] + fx_t(k) * D[a];
                    const long i0 = long((long long)(X >> 64));
                    f[a] = double((unsigned long long)X) * 5.42101086242752217e-20;
                    lo[a] = clampl(i0, 0, N[a] - 1);
                    hi[a] = clampl(i0 + 1, 0, N[a] - 1);
                }
                for (int cc = 0; cc < 8; ++cc) {
                    int dx = (cc >> 2) & 1, dy = (cc >> 1) & 1, dz = cc & 1;
                    corner[k * 8 + cc] = M.cell(dx ? hi[0] : lo[0], dy ? hi[1] : lo[1], dz ? hi[2] : lo[2]);
                    w[k * 8 + cc] = (dx ? f[0] : 1.0 - f[0]) * (dy ? f[1] : 1.0 - f[1]) * (dz ? f[2] : 1.0 - f[2]);
                }
                const size_t base = M.cell(lo[0], lo[1], lo[2]);
                for (long b = 0; b < n_bins; ++b) {
                    const double kap = double(kappa[base + b]);
                    att[k * n_bins + b] = std::exp(-kap * ds);
                    tr[k * n_bins + b] = std::exp(-tau[b]);
                    tau[b] += kap * ds;
                }
            }
            for (long b = 0; b < n_bins; ++b) {                             // backward recurrence
                double lambda = 0.0, a_next = 0.0;
                for (long k = K - 1; k >= 0; --k) {
                    const double* gs = gsuf.data() + size_t(k / Ns) * grid;
                    double G = 0.0;
                    for (int cc = 0; cc < 8; ++cc) G += w[k * 8 + cc] * gs[corner[k * 8 + cc] + b];
                    lambda = scale * G + a_next * lambda;
                    a_next = att[k * n_bins + b];
                    const double v = lambda * tr[k * n_bins + b] * ds;
                    for (int cc = 0; cc < 8; ++cc) acc[t][corner[k * 8 + cc] + b] += w[k * 8 + cc] * v;
                }
            }
        }
    };
    std::vector<std::thread> pool;
    for (long t = 1; t < T; ++t) pool.emplace_back(work, t);
    work(0);
    for (auto& th : pool) th.join();
    for (size_t v = 0; v < grid; ++v) {
        double sum = 0.0;
        for (long u = 0; u < T; ++u) sum += acc[u][v];
        grad_j[v] = sum;
    }
    return 0;
}

// ADJOINT with respect to kappa (the other half of P:64's Jacobian; reading D19).  kappa enters eq. (2)
// through a_k = exp(-kappa_k ds) and T_k = exp(-ds sum_{i<k} kappa_i), kappa_i = kappa[cell of x_i] (nearest
// neighbour, P:29 / D4; the cells do not depend on kappa).  Unrolling eq. (2), I_{k+1} = T_{k+1} sum_{m<=k} ds J_m / a_m
// with J_m = w_m . j, so for L = sum_k G_k I_{k+1}, G_k = s w_k . gsuf[step(k)]:
//     dL/dkappa_i = ds [ ds J_i T_i lambda_{i+1} - R_i ],   R_i = sum_{k >= i} G_k I_{k+1},
// lambda as in rt_adjoint_j_oracle.  Forward sweep recording every substep, then the backward sums, as it reads.
// grad_kappa: double [nx][ny][nz][B], overwritten.
int rt_adjoint_kappa_oracle(const double* gbar, const float* j, const float* kappa, int nx, int ny, int nz,
                            const float* sources, int n_src, int n_rays, int n_bins, float step_size, float c, float dt,
                            int n_steps, double* grad_kappa, int n_threads) {
    if (!gbar || !j || !kappa || !sources || !grad_kappa) return -1;
    if (nx < 1 || ny < 1 || nz < 1 || n_src < 1 || n_rays < 1 || n_bins < 1 || n_steps < 1) return -1;
    if (bad(step_size) || bad(c) || bad(dt)) return -1;
    const long Ns = substeps(double(step_size), double(c), double(dt)), K = Ns * n_steps;
    const double ds = double(step_size);
    const long N[3] = {nx, ny, nz};
    const Medium M{j, kappa, nx, ny, nz, n_bins};
    const size_t grid = size_t(nx) * ny * nz * n_bins;
    const double scale = double(4.0L * kPiL / (long double)n_rays);
    std::vector<double> gsuf(gbar, gbar + grid * size_t(n_steps));
    for (long m = n_steps - 2; m >= 0; --m)
        for (size_t v = 0; v < grid; ++v) gsuf[size_t(m) * grid + v] += gsuf[size_t(m + 1) * grid + v];
    const long total_rays = long(n_src) * n_rays;
    const long T = std::min<long>(std::max(1, n_threads), total_rays);
    std::vector<std::vector<double>> acc(T);
    for (auto& a : acc) a.assign(grid, 0.0);
    auto work = [&](long t) {
        std::vector<size_t> corner(size_t(K) * 8), cell(K);
        std::vector<double> w(size_t(K) * 8), att(K), tr(K), Inext(K), Jv(K);
        for (long r = total_rays * t / T; r < total_rays * (t + 1) / T; ++r) {
            const long s = r / n_rays, i = r % n_rays;
            double nhat[3];
            fib_direction(i, n_rays, nhat);
            fx_t X0[3], D[3];
            for (int a = 0; a < 3; ++a) {
                X0[a] = fx(double(sources[3 * s + a]));
                volatile double step = ds * nhat[a];
                D[a] = fx(step);
            }
            for (long b = 0; b < n_bins; ++b) {
                double I = 0.0, tau = 0.0;
                for (long k = 0; k < K; ++k) {                              // forward sweep, eq. (2)
                    long lo[3], hi[3];
                    double f[3];
                    for (int a = 0; a < 3; ++a) {
                        const fx_t X = X0[a] + fx_t(k) * D[a];
                        const long i0 = long((long long)(X >> 64));
                        f[a] = double((unsigned long long)X) * 5.42101086242752217e-20;
                        lo[a] = clampl(i0, 0, N[a] - 1);
                        hi[a] = clampl(i0 + 1, 0, N[a] - 1);
                    }
                    double jv = 0.0;
                    for (int cc = 0; cc < 8; ++cc) {
                        int dx = (cc >> 2) & 1, dy = (cc >> 1) & 1, dz = cc & 1;
                        corner[k * 8 + cc] = M.cell(dx ? hi[0] : lo[0], dy ? hi[1] : lo[1], dz ? hi[2] : lo[2]);
                        w[k * 8 + cc] = (dx ? f[0] : 1.0 - f[0]) * (dy ? f[1] : 1.0 - f[1]) * (dz ? f[2] : 1.0 - f[2]);
                        jv += w[k * 8 + cc] * double(j[corner[k * 8 + cc] + b]);
                    }
                    cell[k] = M.cell(lo[0], lo[1], lo[2]);
                    const double kap = double(kappa[cell[k] + b]);
                    att[k] = std::exp(-kap * ds);
                    tr[k] = std::exp(-tau);
                    Jv[k] = jv;
                    I = I * att[k] + jv * tr[k] * ds;
                    tau += kap * ds;
                    Inext[k] = I;
                }
                double lambda = 0.0, a_next = 0.0, R = 0.0;
                for (long k = K - 1; k >= 0; --k) {                         // backward sums
                    const double* gs = gsuf.data() + size_t(k / Ns) * grid;
                    double G = 0.0;
                    for (int cc = 0; cc < 8; ++cc) G += w[k * 8 + cc] * gs[corner[k * 8 + cc] + b];
                    G *= scale;
                    lambda = G + a_next * lambda;
                    a_next = att[k];
                    R += G * Inext[k];
                    acc[t][cell[k] + b] += ds * (ds * Jv[k] * tr[k] * lambda - R);
                }
            }
        }
    };
    std::vector<std::thread> pool;
    for (long t = 1; t < T; ++t) pool.emplace_back(work, t);
    work(0);
    for (auto& th : pool) th.join();
    for (size_t v = 0; v < grid; ++v) {
        double sum = 0.0;
        for (long u = 0; u < T; ++u) sum += acc[u][v];
        grad_kappa[v] = sum;
    }
    return 0;
}

// FORWARD-MODE derivative of the march with respect to kappa (gradients "from jacfwd", extending to "a global
// kappa scale"; reading D21): the tangent of the field for kappa -> kappa + eps dkappa at eps = 0 (a global
// scale is dkappa = kappa).  kappa enters eq. (2) through exp(-kappa_k ds) and exp(-tau_k), read nearest
// neighbour at the cell of x_k; the cells do not depend on kappa.  Differentiating eq. (2) term by term,
// with dot = d/d eps:
//   Idot_{k+1}   = Idot_k exp(-kappa_k ds) + I_k (-dkappa_k ds) exp(-kappa_k ds) + j(x_k) (-taudot_k) exp(-tau_k) ds
//   taudot_{k+1} = taudot_k + dkappa_k ds
// next to eq. (2) itself for (I, tau); the tangent field collects w_c Idot_{k+1} with the weights of x_k,
// cumulative snapshots (D7), scaled by 4 pi / N_Omega (D8).  tangent: double [n_steps][nx][ny][nz][B], overwritten.
int rt_jvp_kappa_oracle(const float* j, const float* kappa, const float* dkappa, int nx, int ny, int nz,
                        const float* sources, int n_src, int n_rays, int n_bins, float step_size, float c, float dt,
                        int n_steps, double* tangent, int n_threads) {
    if (!j || !kappa || !dkappa || !sources || !tangent) return -1;
    if (nx < 1 || ny < 1 || nz < 1 || n_src < 1 || n_rays < 1 || n_bins < 1 || n_steps < 1) return -1;
    if (bad(step_size) || bad(c) || bad(dt)) return -1;
    const long Ns = substeps(double(step_size), double(c), double(dt));
    const double ds = double(step_size);
    const long N[3] = {nx, ny, nz};
    const Medium M{j, kappa, nx, ny, nz, n_bins};
    const size_t grid = size_t(nx) * ny * nz * n_bins;
    const double scale = double(4.0L * kPiL / (long double)n_rays);
    const long total_rays = long(n_src) * n_rays;
    const long T = std::min<long>(std::max(1, n_threads), total_rays);
    std::vector<std::vector<double>> acc(T);                  // per thread: [n_steps][grid], per-step increments
    for (auto& a : acc) a.assign(grid * size_t(n_steps), 0.0);
    auto work = [&](long t) {
        for (long r = total_rays * t / T; r < total_rays * (t + 1) / T; ++r) {
            const long s = r / n_rays, i = r % n_rays;
            double nhat[3];
            fib_direction(i, n_rays, nhat);
            fx_t X0[3], D[3];
            for (int a = 0; a < 3; ++a) {
                X0[a] = fx(double(sources[3 * s + a]));
                volatile double step = ds * nhat[a];
                D[a] = fx(step);
            }
            for (long b = 0; b < n_bins; ++b) {
                double I = 0.0, tau = 0.0, Idot = 0.0, taudot = 0.0;
                for (long k = 0; k < Ns * n_steps; ++k) {
                    long lo[3], hi[3];
                    double f[3];
                    for (int a = 0; a < 3; ++a) {
                        const fx_t X = X0[a] + fx_t(k) * D[a];
                        const long i0 = long((long long)(X >> 64));
                        f[a] = double((unsigned long long)X) * 5.42101086242752217e-20;
                        lo[a] = clampl(i0, 0, N[a] - 1);
                        hi[a] = clampl(i0 + 1, 0, N[a] - 1);
                    }
                    size_t corner[8];
                    double w[8], jv = 0.0;
                    for (int cc = 0; cc < 8; ++cc) {
                        int dx = (cc >> 2) & 1, dy = (cc >> 1) & 1, dz = cc & 1;
                        corner[cc] = M.cell(dx ? hi[0] : lo[0], dy ? hi[1] : lo[1], dz ? hi[2] : lo[2]);
                        w[cc] = (dx ? f[0] : 1.0 - f[0]) * (dy ? f[1] : 1.0 - f[1]) * (dz ? f[2] : 1.0 - f[2]);
                        jv += w[cc] * double(j[corner[cc] + b]);
                    }
                    const size_t base = M.cell(lo[0], lo[1], lo[2]);
                    const double kap = double(kappa[base + b]), dkap = double(dkappa[base + b]);
                    const double att = std::exp(-kap * ds), tr = std::exp(-tau);
                    Idot = Idot * att + I * (-dkap * ds) * att + jv * (-taudot) * tr * ds;
                    I = I * att + jv * tr * ds;                              // eq. (2)
                    taudot += dkap * ds;
                    tau += kap * ds;
                    double* slice = acc[t].data() + size_t(k / Ns) * grid;
                    for (int cc = 0; cc < 8; ++cc) slice[corner[cc] + b] += w[cc] * Idot;
                }
            }
        }
    };
    std::vector<std::thread> pool;
    for (long t = 1; t < T; ++t) pool.emplace_back(work, t);
    work(0);
    for (auto& th : pool) th.join();
    for (size_t v = 0; v < grid; ++v) {
        double run = 0.0;
        for (long m = 0; m < n_steps; ++m) {
            for (long u = 0; u < T; ++u) run += acc[u][size_t(m) * grid + v];
            tangent[size_t(m) * grid + v] = scale * run;
        }
    }
    return 0;
}

const char* rt_oracle_version(void) { return "rt_oracle 1 (fp64, PAPER.md eq. 2)"; }

}  // extern "C"
