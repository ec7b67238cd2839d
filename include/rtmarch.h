/* rtmarch.h — C ABI of librtmarch.so: the time-dependent emission-absorption ray march of
 * Ray-trax (arXiv 2511.09389), hand-written CUDA for sm_100a (NVIDIA B200).
 *
 * Citations: P:<n> = line n of the paper text; D<n> = reading n in DESIGN.md §4.
 *
 * WHAT rt_march COMPUTES (eq. (2) at P:23).  For every source s, every direction i of an
 * N_Omega-point Fibonacci (golden-angle) lattice (D1) and every frequency bin b, a ray starts
 * at x_0 = sources[s] with I_0 = tau_0 = 0 (D11) and takes n_steps * N_s substeps, N_s = ceil(c dt / ds)
 * (D6).  Substep k, at x_k = x_0 + k ds n_i (D3):
 *     kappa_b = kappa at the base cell floor(x_k), nearest neighbour, clamped            (D4, D5)
 *     j_b     = trilinear read of j at x_k, indices clamped to the domain                (D5)
 *     I_b   <- I_b exp(-kappa_b ds) + j_b exp(-tau_b) ds ;  tau_b <- tau_b + kappa_b ds  (eq. 2)
 *     field[corner_c][b] += w_c I_b  for the 8 corners, with the SAME trilinear weights  (D2)
 * out[m] is the field after (m+1) N_s substeps (cumulative snapshots, D7), summed over sources
 * and scaled once by 4 pi / N_Omega (D8).
 *
 * LAYOUT.  j, kappa: [nx][ny][nz][n_bins] float32, C order, bin innermost; kappa in 1/cell-length.
 * sources: [n_src][3] float32 grid coordinates (axis 0, 1, 2); voxel (a,b,c) sits at coordinate (a,b,c).
 * out: [n_steps][nx][ny][nz][n_bins] float32, OVERWRITTEN.  j must be finite (a weight-0 corner is still read).  Directions map to axes (0,1,2) as
 * (sqrt(1-z^2) cos phi, sqrt(1-z^2) sin phi, z).
 *
 * POINTERS AND OWNERSHIP.  Unless a function says "host", every pointer is a DEVICE pointer on the current
 * CUDA device, owned by the caller (e.g. a torch tensor's data_ptr()); the library never frees or keeps
 * it.  rt_march* are ASYNCHRONOUS: all work is enqueued on `stream` (a cudaStream_t passed as void*; NULL =
 * the legacy default stream) and the caller synchronises.  j, kappa, sources, out and workspace must not
 * overlap.  Re-entrant per stream (each concurrent call needs its own workspace and out); the only state the
 * library keeps between calls is rt_march_host's memory pool (below) and a thread-local CUDA error string.
 *
 * ERRORS.  Functions returning int give RT_OK (0) or a negative RT_E* code; rt_strerror() names it.
 * Argument errors are detected on the host BEFORE any CUDA call, so they can be exercised without a GPU.
 * Source positions may be any finite value (a source outside the box is legal: clamping defines the
 * result); they are saturated to +-2^29 cells.  Non-finite positions give an unspecified field.
 *
 * LIMITS (RT_EINVAL otherwise): nx*ny*nz*n_bins < 2^31; n_steps*N_s < 2^31; n_steps*N_s*step_size <= 2^28
 * cells; n_rays <= 2^30.
 */
#ifndef RTMARCH_H
#define RTMARCH_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define RT_OK 0
#define RT_EINVAL (-1)     /* null pointer, non-positive size, non-finite / non-positive step_size, c or dt, limit exceeded */
#define RT_EWORKSPACE (-2) /* workspace is NULL or smaller than rt_workspace_bytes() */
#define RT_ECUDA (-3)      /* a CUDA runtime call or kernel launch failed; rt_strerror(RT_ECUDA) holds the CUDA message */
#define RT_EALIGN (-4)     /* j, kappa or out not 4-byte aligned */
#define RT_ETOOBIG (-5)    /* rt_march_static: the call needs more scratch than RT_STATIC_WORKSPACE_BYTES */

/* Kernel variants for rt_march_ex (tests and bench only; rt_march always uses RT_VARIANT_DEFAULT).
 * All variants compute the same field; they differ in how the deposit of P:29 is issued and in which rays
 * share a warp.  A variant code is one kind (0..5), optionally OR-ed with flags. */
#define RT_VARIANT_DEFAULT 0 /* sliding-stencil register accumulation, coherent ray order; warp = 32 sources x 1
                                direction when n_src >= 32, else 32 directions of one source */
#define RT_VARIANT_DIRECT 1  /* textbook form: 8 reductions per ray-substep-bin-group, lattice order */
#define RT_VARIANT_DIRECT_COHERENT 2 /* 8 reductions per ray-substep, coherent ray order */
#define RT_VARIANT_SLIDING_LATTICE 3 /* sliding stencil, rays in lattice-index order, warp = 32 directions */
#define RT_VARIANT_SLIDING_BY_DIRECTION 4 /* sliding stencil, coherent ray order, warp = 32 directions of one source */
#define RT_VARIANT_SLIDING_BY_SOURCE 5 /* sliding stencil, coherent ray order, warp = 32 sorted sources x 1 direction */
#define RT_VARIANT_FLAG_ACC_F32 16 /* accumulate straight into `out` in fp32 instead of the fp64 workspace grid */
#define RT_VARIANT_FLAG_ONE_BIN 32 /* one bin per thread even when n_bins % 4 == 0 (bins in adjacent lanes) */

/* The multi-source march ("loop-and-sum wrapper").  See the header comment for semantics. */
int rt_march(const float* j, const float* kappa, int nx, int ny, int nz,
             const float* sources, int n_src, int n_rays /* N_Omega */, int n_bins,
             float step_size /* ds, cells */, float c /* radiation velocity */, float dt /* time step */,
             int n_steps, float* out,
             void* workspace, size_t workspace_bytes, /* device scratch, >= rt_workspace_bytes(), 16-byte aligned */
             void* stream);

/* rt_march for callers that may not allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the same march (the product kernels of rt_march), its workspace a
 * file-scope __device__ array inside the library instead of a caller's buffer.  The call allocates nothing: no
 * cudaMalloc / cudaFree, no memory pool, no allocating library routine -- it looks the array's device address up
 * (cudaGetSymbolAddress, once per device, with the caller's current device) and enqueues memsets and kernels on
 * `stream` like rt_march.  j, kappa, sources, out: DEVICE pointers on the current device, owned by the caller, rules
 * and limits as rt_march; asynchronous.
 *   LIMIT: rt_workspace_bytes(nx, ny, nz, n_src, n_rays, n_bins, n_steps) <= RT_STATIC_WORKSPACE_BYTES = 96 MiB
 *   (e.g. 128^3 x 1 bin x 1 time step with 2,097 sources: 80.5 MiB; 64^3 x 4 bins x 4 steps: 48 MiB), else
 *   RT_ETOOBIG, returned before any CUDA call.  Every GPU that loads the library holds the array until the process
 *   exits.
 *   SHARED STATE: every rt_march_static call on a device uses the same array, which keeps the last call's contents.
 *   Each call zeroes what it sums into and rebuilds its tables on the stream, so calls that follow each other on one
 *   stream (or are otherwise ordered on the GPU) are independent; calls that OVERLAP on the GPU -- two streams, two
 *   host threads on one device -- race on the array and give wrong fields.  Use rt_march with private workspaces there. */
#define RT_STATIC_WORKSPACE_BYTES (96u << 20)
size_t rt_static_workspace_bytes(void); /* = RT_STATIC_WORKSPACE_BYTES; host only */
int rt_march_static(const float* j, const float* kappa, int nx, int ny, int nz,
                    const float* sources, int n_src, int n_rays, int n_bins,
                    float step_size, float c, float dt, int n_steps, float* out, void* stream);

/* rt_march with kappa read by TRILINEAR interpolation at x_k, with the weights of the j read, instead of nearest
 * neighbour (reading D18: P:29 calls nearest neighbour the current choice).  Everything else as rt_march. */
int rt_march_trilinear_kappa(const float* j, const float* kappa, int nx, int ny, int nz,
                             const float* sources, int n_src, int n_rays, int n_bins,
                             float step_size, float c, float dt, int n_steps, float* out,
                             void* workspace, size_t workspace_bytes, void* stream);

/* The paper's single-source kernel: rt_march with n_src = 1; source_pos = 3 floats (device). */
int rt_march_single(const float* j, const float* kappa, int nx, int ny, int nz,
                    const float* source_pos, int n_rays, int n_bins,
                    float step_size, float c, float dt, int n_steps, float* out,
                    void* workspace, size_t workspace_bytes, void* stream);

/* rt_march with an explicit kernel variant (RT_VARIANT_*).  Unknown variant -> RT_EINVAL. */
int rt_march_ex(const float* j, const float* kappa, int nx, int ny, int nz,
                const float* sources, int n_src, int n_rays, int n_bins,
                float step_size, float c, float dt, int n_steps, float* out,
                void* workspace, size_t workspace_bytes, void* stream, int variant);

/* STEPPING WITH PERSISTENT RAY STATE ("for strict time integration we fix dt and iterate"; P:58 RT substeps
 * between hydro updates; reading D17).  rt_march_step advances every ray by ONE time step -- substeps
 * k_begin .. k_begin + N_s - 1 -- in the medium (j, kappa) passed to THIS call, which the caller may change
 * between calls.  Rays continue their straight lines (x_k = x_0 + k ds n: pass k_begin = m * N_s for step m, with
 * the same sources, n_rays, step_size, c, dt); (I, exp(-tau)) of every (source, direction, bin) carry over in
 * `state`.  out[nx][ny][nz][n_bins] receives the field deposited during this step, scaled by 4 pi / N_Omega:
 * overwritten (accumulate = 0) or added to (accumulate != 0; summed in fp64, rounded once per call).  With an
 * unchanged medium, steps 0..m accumulated reproduce snapshot m of rt_march.
 *   state: device, rt_state_bytes() bytes, 16-byte aligned, float32 [2][n_src][n_rays][n_bins] = I then exp(-tau);
 *          rt_state_reset() gives the fresh state I = 0, tau = 0 (D11).  Indexed by source and lattice index.
 *   workspace: rt_step_workspace_bytes() bytes.  Errors and limits as rt_march, with n_steps*N_s -> k_begin + N_s. */
size_t rt_state_bytes(int n_src, int n_rays, int n_bins);
int rt_state_reset(float* state, int n_src, int n_rays, int n_bins, void* stream);
size_t rt_step_workspace_bytes(int nx, int ny, int nz, int n_src, int n_rays, int n_bins);
int rt_march_step(const float* j, const float* kappa, int nx, int ny, int nz,
                  const float* sources, int n_src, int n_rays, int n_bins,
                  float step_size, float c, float dt, long long k_begin, float* state,
                  float* out, int accumulate, void* workspace, size_t workspace_bytes, void* stream);

/* ADJOINT WITH RESPECT TO j (P:62-64 differentiability; reading D19).  For fixed kappa the field of
 * rt_march is linear in j: out[m] = A_m j.  Given gbar[n_steps][nx][ny][nz][n_bins] = dL/d out[m] (device, fp32)
 * this writes grad_j[nx][ny][nz][n_bins] = sum_m A_m^T gbar[m] = dL/dj (device, fp32, OVERWRITTEN; summed in fp64 -- with
 * one bin through the fp32 scratch of the forward march, drained into the fp64 grid during the march):
 * the backward recurrence of eq. (2), marched along every ray from its last substep to its first with the same
 * clamped trilinear stencils, gather and deposit exchanged.  <rt_march(j), gbar> = <j, grad_j> up to rounding.
 * kappa is read nearest neighbour (as rt_march).  Same argument rules, limits and error codes as rt_march;
 * workspace: rt_adjoint_workspace_bytes() bytes. */
size_t rt_adjoint_workspace_bytes(int nx, int ny, int nz, int n_src, int n_rays, int n_bins, int n_steps);
int rt_march_adjoint_j(const float* gbar, const float* kappa, int nx, int ny, int nz,
                       const float* sources, int n_src, int n_rays, int n_bins,
                       float step_size, float c, float dt, int n_steps, float* grad_j,
                       void* workspace, size_t workspace_bytes, void* stream);

/* ADJOINT WITH RESPECT TO kappa (the other half of P:64's Jacobian; reading D19).  Writes
 * grad_kappa[nx][ny][nz][n_bins] = dL/dkappa (device, fp32, OVERWRITTEN; summed in fp64) for gbar[m] = dL/d out[m] of
 * rt_march(j, kappa, ...): kappa enters eq. (2) through exp(-kappa ds) and exp(-tau), read nearest neighbour at the
 * cell of x_k, so dL/dkappa_i = ds [P_i lambda_{i+1} - sum_{k>=i} G_k I_{k+1}] summed into that cell.  The forward
 * intensities I_{k+1} are recorded (4 bytes per ray-substep-bin; P_i = I_{i+1} - exp(-kappa_i ds) I_i is recovered from them; sources in batches so the record stays below 8 GiB) and the
 * rays are then marched backwards.  Same argument rules, limits and error codes as rt_march; workspace:
 * rt_adjoint_kappa_workspace_bytes() bytes (0 on invalid arguments). */
size_t rt_adjoint_kappa_workspace_bytes(int nx, int ny, int nz, int n_src, int n_rays, int n_bins,
                                        float step_size, float c, float dt, int n_steps);
int rt_march_adjoint_kappa(const float* gbar, const float* j, const float* kappa, int nx, int ny, int nz,
                           const float* sources, int n_src, int n_rays, int n_bins,
                           float step_size, float c, float dt, int n_steps, float* grad_kappa,
                           void* workspace, size_t workspace_bytes, void* stream);

/* FORWARD-MODE DERIVATIVE WITH RESPECT TO kappa (gradients "from jacfwd", "a global kappa scale"; DESIGN.md
 * reading D21).  Writes tangent[n_steps][nx][ny][nz][n_bins] = d/d eps of rt_march(j, kappa + eps dkappa, ...) at eps = 0
 * (device, fp32, OVERWRITTEN; cumulative snapshots like out).  dkappa has kappa's shape and layout; a global scale
 * kappa -> theta kappa is dkappa = kappa.  The tangent of eq. (2) -- Idot_{k+1} = a_k (Idot_k - I_k dkappa_k ds) - j(x_k)
 * taudot_k exp(-tau_k) ds, taudot_{k+1} = taudot_k + dkappa_k ds, kappa and dkappa read at the cell of x_k -- is marched
 * next to eq. (2) and deposited with the weights of x_k.  <gbar, tangent> = <rt_march_adjoint_kappa(gbar), dkappa> up to
 * rounding.  Argument rules, limits, error codes and workspace (rt_workspace_bytes) as rt_march, and step_size must be
 * below one cell (RT_EINVAL otherwise). */
int rt_march_jvp_kappa(const float* j, const float* kappa, const float* dkappa, int nx, int ny, int nz,
                       const float* sources, int n_src, int n_rays, int n_bins,
                       float step_size, float c, float dt, int n_steps, float* tangent,
                       void* workspace, size_t workspace_bytes, void* stream);

/* TEST HOOK.  rt_march_adjoint_kappa with the bound on the forward record of one source batch given explicitly
 * (record_limit bytes; 0 = the library's 8 GiB), so that tests can drive the source-batch loop on small cases.  A batch
 * never holds fewer than 32 sources (n_src >= 32) or 1 source (n_src < 32).  Same result for every limit. */
size_t rt_adjoint_kappa_workspace_bytes_ex(int nx, int ny, int nz, int n_src, int n_rays, int n_bins,
                                           float step_size, float c, float dt, int n_steps, size_t record_limit);
int rt_march_adjoint_kappa_ex(const float* gbar, const float* j, const float* kappa, int nx, int ny, int nz,
                              const float* sources, int n_src, int n_rays, int n_bins,
                              float step_size, float c, float dt, int n_steps, float* grad_kappa,
                              void* workspace, size_t workspace_bytes, void* stream, size_t record_limit);

/* End-to-end form with HOST pointers (j, kappa, sources, out are host memory, pinned or pageable).
 * Allocates device buffers, copies the inputs in, marches, copies out[] back, frees, and returns after the
 * copy has completed (SYNCHRONOUS).  Same semantics, limits and error codes as rt_march.  The device buffers come
 * from a private stream-ordered memory pool per device that keeps its memory between calls (the library's only
 * retained state); rt_host_release() gives it back. */
int rt_march_host(const float* j, const float* kappa, int nx, int ny, int nz,
                  const float* sources, int n_src, int n_rays, int n_bins,
                  float step_size, float c, float dt, int n_steps, float* out);

int rt_host_release(void);

/* Bytes of device scratch one rt_march call needs: the ray-order and source-order tables, the fp64 accumulation grid
 * (n_steps * nx*ny*nz*n_bins doubles: deposits are summed in fp64 and rounded to fp32 once; the kernels
 * of the non-default variants spread their reductions over up to 4 copies of it where they fit 48 MiB), one fp32 grid
 * of n_steps * nx*ny*nz*n_bins floats where the batched multi-bin kernels of the variants run (n_bins % 4 == 0 and that
 * grid <= 128 MiB), for one-bin calls the fp32 window-brick scratch of the march (n_steps * nx*(ny+1)*(nz+1)*4
 * floats, if <= 1 GiB), and for grids far larger than the L2 (that fp32 grid > 128 MiB, no brick scratch,
 * n_src * n_rays < 2^32) the sorted ray list (8 bytes per ray + 4 MiB, and with bins in fours a ray state of
 * 8 bytes per ray and bin).  0 on invalid arguments. */
size_t rt_workspace_bytes(int nx, int ny, int nz, int n_src, int n_rays, int n_bins, int n_steps);

/* N_s as the library computes it (D6): ceil(c dt / step_size), a ratio within 1e-6 (relative) of an
 * integer counts as that integer.  Host only.  Returns RT_EINVAL on non-finite or non-positive input, or if
 * N_s >= 2^31. */
int rt_substeps_per_step(float step_size, float c, float dt);

/* Number of kernels of this library that one rt_march call with these arguments and a step_size below one cell
 * enqueues (memsets excluded).  Calls that march from the sorted ray list (rt_workspace_bytes) enqueue 5 -- key,
 * prefix sums, scatter, march, snapshots -- or, with bins in fours and few deposits per element, 7:
 * + ray-state reset and a second march launch; 7 is returned whenever the bins come in fours. */
int rt_launch_count(int nx, int ny, int nz, int n_src, int n_rays, int n_bins, int n_steps);

/* TEST HOOK.  Writes the library's direction lattice (D1) for i = 0..n_rays-1 into
 * nhat[n_rays][3] (float64, device), computed exactly as the march kernel does. */
int rt_directions(int n_rays, double* nhat, void* stream);

/* TEST HOOK.  Marches ONE ray (source_pos[3], lattice index ray_index of n_rays) for n_sub substeps from k = 0
 * with the arithmetic of the march kernels (fixed-point position, fp32 weights, gather, eq. (2)) and records,
 * per substep k: pos[k][3] = x_k (float64), trace_I[k][b] = I_{k+1} (NOT scaled by 4 pi/N_Omega) and
 * trace_T[k][b] = exp(-tau_{k+1}).  All pointers device; nothing is deposited. */
int rt_trace_ray(const float* j, const float* kappa, int nx, int ny, int nz, int n_bins,
                 const float* source_pos, int ray_index, int n_rays, float step_size, int n_sub,
                 double* pos, float* trace_I, float* trace_T, void* stream);

/* TEST HOOK.  Writes the coherent ray order into order[rt_ray_slots(n_rays)] (uint32, device): slot ->
 * lattice index, 0xFFFFFFFF for padding slots.  Every index 0..n_rays-1 appears exactly once. */
int rt_ray_order(int n_rays, unsigned int* order, void* stream);
int rt_ray_slots(int n_rays);

/* BENCH ONLY: reduction-throughput ceilings ("measured L2-atomic roofline").  Issues
 * `n_red` (rounded up to a whole number per thread; the exact count issued is returned through
 * *n_issued, host pointer, may be NULL) fp32 reductions into grid[nx][ny][nz][n_bins] on `stream`:
 *   mode 0  scalar red.global.add.f32, uniformly random addresses                         (M1)
 *   mode 1  red.global.add.v4.f32, uniformly random 16-byte-aligned addresses             (M2)
 *   mode 2  trilinear-stencil pattern: random base voxel, its 8 corners; scalar reds when
 *           n_bins % 4 != 0, else n_bins/4 v4 reds per corner                             (M3 = R*)
 *   mode 3  every reduction to one address                                                (M4)
 *   mode 4  warp-coalesced: 32 consecutive floats per warp instruction, random line       (M5)
 *   mode 5  M3 issued along a random walk of half a cell per step (ray-like locality)     (M6)
 *   mode 6  scalar red.global.add.f64, uniformly random addresses                         (M1 in fp64)
 *   mode 7  the stencil pattern of mode 2 with n_bins scalar red.global.add.f64 per corner (M3 in fp64)
 *   mode 8  scalar reds spread over the 8 corner voxels of the grid                          (M4, 8 addresses)
 *   mode 9  scalar reds to uniformly random voxels of the boundary shell                     (M4, shell)
 * `grid` holds nx*ny*nz*n_bins floats (modes 0-5, 8, 9) or doubles (modes 6, 7).
 * The grid is only accumulated into (caller zero-fills if the content matters). */
int rt_bench_red_ceiling(int mode, void* grid, int nx, int ny, int nz, int n_bins,
                         long long n_red, unsigned int seed, long long* n_issued, void* stream);

const char* rt_strerror(int code);
const char* rt_version(void);

#ifdef __cplusplus
}
#endif
#endif /* RTMARCH_H */
