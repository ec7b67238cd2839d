"""Pins for the fp64 oracle (oracle/rt_oracle.cpp): what the paper and the mathematics fix.

Every test here checks the oracle against something that is NOT the oracle: 50-digit arithmetic, closed
forms derived from eq. (2), invariants (deposit mass, horizon, linearity), a library routine
(scipy's order-1 map_coordinates) in the special case where the march reduces to it, the analytic point
source of eq. (3), a dense tent-function brute force on tiny non-cubic grids, and traces
unrolled by hand on a 4^3 grid.  P<n> labels follow SURVEY.md §8(c) / DESIGN.md §6.
"""
import math

import numpy as np
import pytest

import workloads as W

FOUR_PI = 4.0 * math.pi


def f32(x):
    return float(np.float32(x))


# ------------------------------------------------------------------------------------------------------
# P0  direction lattice (reading D1) against 50-digit arithmetic
# ------------------------------------------------------------------------------------------------------
def test_p0_directions_match_50_digit_arithmetic(oracle_mod):
    import mpmath as mp
    mp.mp.dps = 50
    golden_angle = mp.pi * (3 - mp.sqrt(5))
    for n in (1, 2, 3, 64, 1024, 4096, 16384):
        idx = sorted(set([0, 1, n // 3, n // 2, n - 2, n - 1]) & set(range(n)))
        for i in idx:
            z = 1 - mp.mpf(2 * i + 1) / n
            s = mp.sqrt(1 - z * z)
            phi = i * golden_angle
            ref = [float(s * mp.cos(phi)), float(s * mp.sin(phi)), float(z)]
            got = oracle_mod.direction(i, n)
            assert np.max(np.abs(got - ref)) < 3e-16, (n, i, got, ref)
    # every index of the largest lattice the configs use: the azimuth reduction must not lose i * eps
    n = 16384
    worst = 0.0
    for i in range(0, n, 7):
        z = 1 - mp.mpf(2 * i + 1) / n
        s = mp.sqrt(1 - z * z)
        phi = i * golden_angle
        ref = [float(s * mp.cos(phi)), float(s * mp.sin(phi)), float(z)]
        worst = max(worst, float(np.max(np.abs(oracle_mod.direction(i, n) - ref))))
    assert worst < 3.5e-16, worst


def test_p0_lattice_is_unit_and_nearly_uniform(oracle_mod):
    n = 4096
    d = np.array([oracle_mod.direction(i, n) for i in range(n)])
    assert np.allclose(np.linalg.norm(d, axis=1), 1.0, atol=1e-15)
    # single direction lattice is the +axis-0 ray (hand-traceable, D1)
    assert np.array_equal(oracle_mod.direction(0, 1), [1.0, 0.0, 0.0])
    # z is an exact midpoint rule on [-1, 1]; first moments vanish, second moments are isotropic
    assert np.allclose(np.sort(d[:, 2]), -1 + (2 * np.arange(n) + 1) / n, atol=1e-15)
    assert np.all(np.abs(d.mean(axis=0)) < 2e-3)
    assert np.allclose(d.T @ d / n, np.eye(3) / 3, atol=2e-3)
    # nearest-neighbour separation ~ sqrt(4 pi / n): no clumps, no duplicates
    sub = d[::8]
    dots = d @ sub.T
    dots[np.arange(0, n, 8), np.arange(sub.shape[0])] = -1
    nn = np.arccos(np.clip(dots.max(axis=0), -1, 1))
    mean_spacing = math.sqrt(FOUR_PI / n)
    assert nn.min() > 0.5 * mean_spacing and nn.max() < 1.5 * mean_spacing


def test_substeps_rule(oracle_mod):
    # PAPER.md:25  N_s = ceil(c dt / ds); all five configs have integer ratios
    assert oracle_mod.substeps(0.5, 1.0, 12.0) == 24
    assert oracle_mod.substeps(0.5, 1.0, 16.0) == 32
    assert oracle_mod.substeps(0.5, 1.0, 222.0) == 444
    assert oracle_mod.substeps(0.5, 1.0, 64.0) == 128
    assert oracle_mod.substeps(0.5, 1.0, 32.0) == 64
    assert oracle_mod.substeps(0.3, 1.0, 1.0) == 4          # 3.33 -> 4
    assert oracle_mod.substeps(1.0, 2.0, 0.75) == 2         # 1.5 -> 2
    assert oracle_mod.substeps(0.1, 1.0, 0.3) == 3          # fp noise in 0.3/0.1 must not give 4
    assert oracle_mod.substeps(2.0, 1.0, 1.0) == 1
    assert oracle_mod.substeps(-1.0, 1.0, 1.0) == -1


# ------------------------------------------------------------------------------------------------------
# P1  closed form in a uniform medium:  I_k = k j0 ds a^(k-1),  tau_k = k kappa0 ds,  a = exp(-kappa0 ds)
#     (induction on eq. (2) with exp(-tau_k) = a^k)
# ------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("src", [(7.5, 7.5, 7.5), (0.25, 14.0, 3.75), (-3.0, 20.0, 5.0)])
def test_p1_uniform_medium_closed_form(oracle_mod, src):
    j0, k0, ds, nsub = f32(0.3), f32(0.1), 0.5, 40
    j, kap = W.uniform_medium(16, j0, k0)
    a = math.exp(-k0 * ds)
    for ray in (0, 17, 63):
        tr = oracle_mod.trace_ray(j, kap, src, ray, 64, ds, nsub)
        k = np.arange(1, nsub + 1)
        assert np.allclose(tr["I"][:, 0], k * j0 * ds * a ** (k - 1), rtol=1e-13, atol=0)
        assert np.allclose(tr["tau"][:, 0], k * k0 * ds, rtol=1e-13, atol=0)


# ------------------------------------------------------------------------------------------------------
# P2  deposit-mass conservation (BASELINE.json north_star): every substep deposits total weight 1, also
#     when clamped, so  sum(out) = (4 pi/N) sum_rays sum_k I_{k+1}.
# ------------------------------------------------------------------------------------------------------
def test_p2_mass_uniform_medium_closed_form(oracle_mod):
    n, j0, k0, ds, Ns, n_src = 16, f32(0.3), f32(0.1), 0.5, 24, 3
    j, kap = W.uniform_medium(n, j0, k0)
    src = np.array([[7.5, 7.5, 7.5], [1.0, 2.0, 14.5], [15.0, 0.0, 8.25]], np.float32)
    a = math.exp(-k0 * ds)
    # sum_{k=1..Ns} k a^(k-1) = [1 - (Ns+1) a^Ns + Ns a^(Ns+1)] / (1-a)^2
    expect = FOUR_PI * n_src * j0 * ds * (1 - (Ns + 1) * a ** Ns + Ns * a ** (Ns + 1)) / (1 - a) ** 2
    for n_rays in (1, 7, 64):
        out = oracle_mod.march(j, kap, src, n_rays, ds, 1.0, 12.0, 1)
        assert out.sum() == pytest.approx(expect, rel=1e-12)      # also P3: exactly independent of N_Omega
    j, kap = W.uniform_medium(n, j0, 0.0)
    out = oracle_mod.march(j, kap, src, 5, ds, 1.0, 12.0, 1)
    assert out.sum() == pytest.approx(FOUR_PI * n_src * j0 * ds * Ns * (Ns + 1) / 2, rel=1e-12)


def test_p2_per_ray_mass_in_a_random_medium_with_clamping(oracle_mod):
    rng = np.random.default_rng(5)
    shape = (6, 5, 7)
    j = rng.uniform(0.1, 2.0, shape + (2,)).astype(np.float32)
    kap = rng.uniform(0.0, 1.5, shape + (2,)).astype(np.float32)
    for ray in range(11):
        tr = oracle_mod.trace_ray(j, kap, (4.6, 0.3, 5.9), ray, 11, 0.37, 40, deposit=True)
        assert tr["acc"].min() >= 0.0
        for b in range(2):       # sum of deposited weights == 1 per substep  =>  mass == sum_k I_{k+1}
            assert tr["acc"][..., b].sum() == pytest.approx(tr["I"][:, b].sum(), rel=1e-13)
        assert np.abs(tr["pos"][-1] - np.array([4.6, 0.3, 5.9], np.float32)).max() > 2.0   # the ray did leave the box


# ------------------------------------------------------------------------------------------------------
# P3  N_Omega invariance of the 4 pi/N-normalised field
# ------------------------------------------------------------------------------------------------------
def test_p3_total_converges_in_n_omega(oracle_mod):
    n = 32
    rho = W.lognormal_density(n, 11, 1.0)
    j = (1e-3 * rho ** 2)[..., None].astype(np.float32)
    kap = (0.05 * rho)[..., None].astype(np.float32)
    src = np.array([[15.3, 16.1, 14.8]], np.float32)
    tot = [oracle_mod.march(j, kap, src, nr, 0.5, 1.0, 10.0, 1).sum() for nr in (256, 1024, 4096)]
    assert abs(tot[1] / tot[2] - 1) < 2e-3
    assert abs(tot[0] / tot[2] - 1) < 5e-2
    assert abs(tot[1] - tot[2]) <= abs(tot[0] - tot[2])           # monotone convergence


# ------------------------------------------------------------------------------------------------------
# P4  analytic point source, eq. (3):  J(r) = L exp(-kappa r) / (4 pi r^2)
#     Uniform kappa0 gives I_k = a^(k-1) S_k with S_k the Riemann sum of j along the ray; outside the
#     blob S_k = S.  The deposit at x_k (r = k ds) carries I_{k+1} = a^k S = S exp(-kappa0 r), so the field is
#        (4 pi/N) * [N/(ds 4 pi r^2) samples per unit volume] * S exp(-kappa0 r) = S exp(-kappa0 r) / (ds r^2),
#     i.e. eq. (3) with L = 4 pi S / ds.
#     S for a Gaussian blob read trilinearly: the interpolant is the sampled Gaussian convolved with a
#     tent (variance 1/6 per axis), so the radial line integral is A sigma sqrt(pi/2) sigma^2/(sigma^2+1/6),
#     plus the left-endpoint term j(0) ds/2.
# ------------------------------------------------------------------------------------------------------
def _shell_means(field, centre, radii, half_width=0.5):
    ax = [np.arange(s) - c for s, c in zip(field.shape, centre)]
    r = np.sqrt(ax[0][:, None, None] ** 2 + ax[1][None, :, None] ** 2 + ax[2][None, None, :] ** 2)
    return np.array([field[np.abs(r - R) < half_width].mean() for R in radii]), r


def test_p4_point_source_matches_eq3(oracle_mod):
    n, sigma, k0, ds, n_rays = 64, 2.0, f32(0.05), 0.5, 4096
    ctr = (31.5, 31.5, 31.5)
    jb = W.gaussian_blob((n, n, n), ctr, sigma)
    j = jb[..., None].astype(np.float32)
    kap = np.full((n, n, n, 1), k0, np.float32)
    out = oracle_mod.march(j, kap, np.array([ctr], np.float32), n_rays, ds, 1.0, 26.0, 1)[0, ..., 0]
    s2 = sigma * sigma
    amp0 = (s2 / (s2 + 1 / 6)) ** 1.5                      # tent-smoothed central value
    S = sigma * math.sqrt(math.pi / 2) * s2 / (s2 + 1 / 6) + amp0 * ds / 2
    radii = np.arange(11.0, 24.0, 2.0)                     # outside the blob (5.5 sigma), inside the horizon (26)
    mean, _ = _shell_means(out, ctr, radii)
    pred = S * np.exp(-k0 * radii) / (ds * radii ** 2)
    ratio = mean / pred
    assert np.all(np.abs(ratio - 1) < 0.01), ratio          # paper's own figure is 3.16 %
    # shape alone: r^2 exp(kappa r) J(r) is flat to better than 1 %
    flat = mean * radii ** 2 * np.exp(k0 * radii)
    assert flat.max() / flat.min() < 1.01


def test_p4_superposition_of_point_sources(oracle_mod):
    # eq. (3) is a sum over sources: two separated blobs; along the line joining them the field is the sum
    n, sigma, k0, ds = 48, 1.5, f32(0.08), 0.5
    c1, c2 = (13.5, 23.5, 23.5), (34.5, 23.5, 23.5)        # cell-centred, like P4 above
    jb = W.gaussian_blob((n, n, n), c1, sigma) + W.gaussian_blob((n, n, n), c2, sigma)
    j = jb[..., None].astype(np.float32)
    kap = np.full((n, n, n, 1), k0, np.float32)
    src = np.array([c1, c2], np.float32)
    out = oracle_mod.march(j, kap, src, 4096, ds, 1.0, 40.0, 1)[0, ..., 0]
    s2 = sigma * sigma
    S = sigma * math.sqrt(math.pi / 2) * s2 / (s2 + 1 / 6) + (s2 / (s2 + 1 / 6)) ** 1.5 * ds / 2
    # voxels on the mid-plane x = 24 within 6.5 cells of the axis: r1 = r2 there
    ys, zs = np.meshgrid(np.arange(17, 31), np.arange(17, 31), indexing="ij")
    r = np.sqrt(10.5 ** 2 + (ys - 23.5) ** 2 + (zs - 23.5) ** 2)
    pred = 2 * S * np.exp(-k0 * r) / (ds * r ** 2)
    got = out[24, 17:31, 17:31]
    assert abs(got.mean() / pred.mean() - 1) < 0.03
    assert np.median(np.abs(got / pred - 1)) < 0.05          # voxel-wise: percent level, like the paper


def test_p4_error_shrinks_with_more_directions(oracle_mod):
    n, sigma, k0, ds = 48, 2.0, f32(0.05), 0.5
    ctr = (23.5, 23.5, 23.5)
    j = W.gaussian_blob((n, n, n), ctr, sigma)[..., None].astype(np.float32)
    kap = np.full((n, n, n, 1), k0, np.float32)
    s2 = sigma * sigma
    S = sigma * math.sqrt(math.pi / 2) * s2 / (s2 + 1 / 6) + (s2 / (s2 + 1 / 6)) ** 1.5 * ds / 2
    errs = []
    for n_rays in (256, 1024, 4096):
        out = oracle_mod.march(j, kap, np.array([ctr], np.float32), n_rays, ds, 1.0, 20.0, 1)[0, ..., 0]
        _, r = _shell_means(out, ctr, [12.0])
        m = (r > 11) & (r < 18)
        pred = S * np.exp(-k0 * r[m]) / (ds * r[m] ** 2)
        errs.append(np.mean(np.abs(out[m] / pred - 1)))
    assert errs[0] > errs[1] > errs[2]                      # monotone in N_Omega
    assert errs[2] < 0.05


# ------------------------------------------------------------------------------------------------------
# P5  light-front horizon (PAPER.md:13 (i), :21): exactly zero beyond the last deposit + stencil reach
# ------------------------------------------------------------------------------------------------------
def test_p5_horizon_is_exactly_dark(oracle_mod):
    n = 40
    rho = W.lognormal_density(n, 3, 1.0)
    j = (1e-3 * rho ** 2)[..., None].astype(np.float32)
    kap = (0.05 * rho)[..., None].astype(np.float32)
    src = np.array([[12.2, 13.7, 11.1], [27.0, 25.5, 28.3]], np.float32)
    ds, c, dt, n_steps = 0.5, 1.0, 4.0, 3
    Ns = oracle_mod.substeps(ds, c, dt)
    out = oracle_mod.march(j, kap, src, 512, ds, c, dt, n_steps)
    ax = np.arange(n, dtype=np.float64)
    d = np.full((n, n, n), np.inf)
    for s in src.astype(np.float64):
        d = np.minimum(d, np.sqrt((ax[:, None, None] - s[0]) ** 2 + (ax[None, :, None] - s[1]) ** 2
                                  + (ax[None, None, :] - s[2]) ** 2))
    for m in range(n_steps):
        reach = ((m + 1) * Ns - 1) * ds + math.sqrt(3.0)
        assert np.all(out[m, ..., 0][d > reach] == 0.0)
        assert np.all(out[m, ..., 0][d < min(reach - 2.5, 5.0)] > 0.0)      # and lit inside (512 rays: gap-free to r = 5)
        assert np.mean(out[m, ..., 0][d < reach - 2.5] > 0.0) > 0.9
    assert np.all(out[1] >= out[0]) and np.all(out[2] >= out[1])  # cumulative snapshots (D7)


# ------------------------------------------------------------------------------------------------------
# D3  positions on the 2^-64 cell grid (DESIGN.md §4 D3): x_k = (floor(x_0 2^64) + k floor(ds nhat 2^64)) / 2^64.
#     Independent arithmetic: Python exact rationals (fractions.Fraction of the very doubles).  The cases
#     include rays whose exact position lands on an integer plane (z_i rational, N_Omega not a power of two),
#     where floor() -- hence the nearest-neighbour kappa cell -- would otherwise hinge on
#     floating-point rounding order.
# ------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n_rays,ray,src,ds,n_sub", [
    (7, 4, (0.0, 3.0, 2.0), 0.5, 10),          # z = -2/7: exact z-position 1.0 at k = 7
    (33, 7, (0.0, 5.0, 1.5), 0.25, 12),
    (40, 18, (-3.0, 9.0, 2.5), 0.5, 48),
    (5, 0, (1.0, 2.0, 0.0), 0.5, 12),          # nhat = (0.6, 0, 0.8) up to rounding: x hits 4.0 at k = 10
    (64, 11, (7.5, 7.5, 7.5), 0.5, 24),
    (1, 0, (1.0, 1.25, 2.5), 0.5, 8),
])
def test_d3_positions_live_on_the_2_64_grid(oracle_mod, n_rays, ray, src, ds, n_sub):
    from fractions import Fraction
    shape = (6, 5, 4)
    rng = np.random.default_rng(11)
    j = rng.uniform(0.1, 1.0, shape + (1,)).astype(np.float32)
    kap = rng.uniform(0.0, 0.6, shape + (1,)).astype(np.float32)
    tr = oracle_mod.trace_ray(j, kap, src, ray, n_rays, ds, n_sub)
    nh = oracle_mod.direction(ray, n_rays)
    two64 = 1 << 64
    X0 = [math.floor(Fraction(f32(v)) * two64) for v in src]
    D = [math.floor(Fraction(float(f32(ds)) * float(nh[a])) * two64) for a in range(3)]   # ONE double rounding of ds*nhat
    I = tau = 0.0
    dsd = float(f32(ds))
    for k in range(n_sub):
        lo, hi, f = [], [], []
        for a in range(3):
            X = X0[a] + k * D[a]
            i0, frac = X >> 64, X & (two64 - 1)                 # Python's >> floors
            f.append(float(frac) * 2.0 ** -64)
            lo.append(min(max(i0, 0), shape[a] - 1))
            hi.append(min(max(i0 + 1, 0), shape[a] - 1))
            assert abs(tr["pos"][k, a] - (i0 + f[a])) <= 1e-15 * max(1.0, abs(i0))
            assert abs((i0 + f[a]) - (float(f32(src[a])) + k * dsd * nh[a])) < 1e-13
        jv = 0.0
        for c in range(8):
            d = ((c >> 2) & 1, (c >> 1) & 1, c & 1)
            w = 1.0
            for a in range(3):
                w *= f[a] if d[a] else 1.0 - f[a]
            jv += w * float(j[tuple(hi[a] if d[a] else lo[a] for a in range(3))][0])
        kk = float(kap[lo[0], lo[1], lo[2], 0])
        I = I * math.exp(-kk * dsd) + jv * math.exp(-tau) * dsd
        tau += kk * dsd
        assert abs(tr["I"][k, 0] - I) <= 1e-13 * I and abs(tr["tau"][k, 0] - tau) <= 1e-13 * max(tau, 1e-30)


# ------------------------------------------------------------------------------------------------------
# P6  traces unrolled by hand on a 4^3 grid (BASELINE.json north_star).  N_Omega = 1 gives nhat = (1,0,0).
#     These are the only pins for readings D2 (deposit with the weights of x_k), D4 (kappa at the base
#     cell floor(x_k)) and D5 (clamped indices, weights from the unclamped fraction).
# ------------------------------------------------------------------------------------------------------
def _grid4():
    a, b, c = np.meshgrid(np.arange(4), np.arange(4), np.arange(4), indexing="ij")
    J = (1.0 + a + 0.25 * b * b + 0.125 * c + 0.5 * a * c).astype(np.float32)      # distinct per cell
    K = (0.125 + 0.25 * a + 0.0625 * b + 0.03125 * c * c).astype(np.float32)
    return J, K


def test_p6_hand_trace_axis_ray_through_and_out_of_a_4cube(oracle_mod):
    J, K = _grid4()
    J, K = J.astype(np.float64), K.astype(np.float64)
    ds = 0.5
    # source (1, 1.25, 2.5): f_y = .25 -> y cells {1,2} weights {.75,.25}; f_z = .5 -> z cells {2,3} weights {.5,.5}
    def yz(F, x):      # the y-z part of the trilinear read at x-cell `x`
        return 0.75 * 0.5 * F[x, 1, 2] + 0.75 * 0.5 * F[x, 1, 3] + 0.25 * 0.5 * F[x, 2, 2] + 0.25 * 0.5 * F[x, 2, 3]

    dep = np.zeros((4, 4, 4))

    def put(x, wx, I):  # deposit wx * I over the same four (y, z) cells
        dep[x, 1, 2] += wx * 0.75 * 0.5 * I
        dep[x, 1, 3] += wx * 0.75 * 0.5 * I
        dep[x, 2, 2] += wx * 0.25 * 0.5 * I
        dep[x, 2, 3] += wx * 0.25 * 0.5 * I

    exp = math.exp
    # k=0: x=1.0  cell 1, f=0        kappa = K[1,1,2]
    I1 = 0.0 * exp(-K[1, 1, 2] * ds) + yz(J, 1) * exp(-0.0) * ds
    t1 = K[1, 1, 2] * ds
    put(1, 1.0, I1)
    # k=1: x=1.5  cell 1, f=.5       kappa = K[1,1,2] (same base cell)
    I2 = I1 * exp(-K[1, 1, 2] * ds) + (0.5 * yz(J, 1) + 0.5 * yz(J, 2)) * exp(-t1) * ds
    t2 = t1 + K[1, 1, 2] * ds
    put(1, 0.5, I2); put(2, 0.5, I2)
    # k=2: x=2.0  cell 2, f=0        kappa = K[2,1,2]
    I3 = I2 * exp(-K[2, 1, 2] * ds) + yz(J, 2) * exp(-t2) * ds
    t3 = t2 + K[2, 1, 2] * ds
    put(2, 1.0, I3)
    # k=3: x=2.5  cell 2, f=.5
    I4 = I3 * exp(-K[2, 1, 2] * ds) + (0.5 * yz(J, 2) + 0.5 * yz(J, 3)) * exp(-t3) * ds
    t4 = t3 + K[2, 1, 2] * ds
    put(2, 0.5, I4); put(3, 0.5, I4)
    # k=4: x=3.0  cell 3, f=0; upper index 4 clamps to 3
    I5 = I4 * exp(-K[3, 1, 2] * ds) + yz(J, 3) * exp(-t4) * ds
    t5 = t4 + K[3, 1, 2] * ds
    put(3, 1.0, I5)
    # k=5: x=3.5  cell 3, f=.5; both indices are 3 -> all weight on x=3
    I6 = I5 * exp(-K[3, 1, 2] * ds) + (0.5 * yz(J, 3) + 0.5 * yz(J, 3)) * exp(-t5) * ds
    t6 = t5 + K[3, 1, 2] * ds
    put(3, 0.5, I6); put(3, 0.5, I6)
    # k=6: x=4.0  outside: cell 4 clamps to 3; the ray keeps emitting/attenuating with boundary values
    I7 = I6 * exp(-K[3, 1, 2] * ds) + yz(J, 3) * exp(-t6) * ds
    t7 = t6 + K[3, 1, 2] * ds
    put(3, 1.0, I7)
    # k=7: x=4.5
    I8 = I7 * exp(-K[3, 1, 2] * ds) + yz(J, 3) * exp(-t7) * ds
    t8 = t7 + K[3, 1, 2] * ds
    put(3, 1.0, I8)

    j4, k4 = _grid4()
    tr = oracle_mod.trace_ray(j4[..., None], k4[..., None], (1.0, 1.25, 2.5), 0, 1, ds, 8, deposit=True)
    assert np.allclose(tr["pos"][:, 0], 1.0 + 0.5 * np.arange(8), atol=0) and np.all(tr["pos"][:, 1] == 1.25)
    assert np.allclose(tr["I"][:, 0], [I1, I2, I3, I4, I5, I6, I7, I8], rtol=1e-14, atol=0)
    assert np.allclose(tr["tau"][:, 0], [t1, t2, t3, t4, t5, t6, t7, t8], rtol=1e-14, atol=0)
    assert np.allclose(tr["acc"][..., 0], dep, rtol=1e-14, atol=1e-300)
    # the full call: N_Omega = 1, one step of 8 substeps, scaled by 4 pi / 1
    out = oracle_mod.march(j4[..., None], k4[..., None], np.array([[1.0, 1.25, 2.5]], np.float32), 1, ds, 1.0,
                           4.0, 1)
    assert np.allclose(out[0, ..., 0], FOUR_PI * dep, rtol=1e-14, atol=1e-300)


def test_p6_hand_trace_oblique_ray_n_omega_2(oracle_mod):
    # N_Omega = 2, ray 0: z = 1/2, phi = 0  =>  nhat = (sqrt(3)/2, 0, 1/2).  Source (0.5, 2, 0.5), ds = 1.
    J, K = _grid4()
    J, K = J.astype(np.float64), K.astype(np.float64)
    r3 = math.sqrt(3.0) / 2
    exp = math.exp
    dep = np.zeros((4, 4, 4))
    # k=0: p = (0.5, 2, 0.5): cells (0,2,0), f = (.5, 0, .5)
    jv = 0.25 * (J[0, 2, 0] + J[0, 2, 1] + J[1, 2, 0] + J[1, 2, 1])
    I1 = jv * 1.0
    t1 = K[0, 2, 0] * 1.0
    for (x, z) in ((0, 0), (0, 1), (1, 0), (1, 1)):
        dep[x, 2, z] += 0.25 * I1
    # k=1: p = (0.5 + r3, 2, 1.0) = (1.3660.., 2, 1): cells (1,2,1), f = (r3 - .5, 0, 0)
    fx = r3 - 0.5
    jv = (1 - fx) * J[1, 2, 1] + fx * J[2, 2, 1]
    I2 = I1 * exp(-K[1, 2, 1]) + jv * exp(-t1)
    t2 = t1 + K[1, 2, 1]
    dep[1, 2, 1] += (1 - fx) * I2
    dep[2, 2, 1] += fx * I2
    # k=2: p = (0.5 + 2 r3, 2, 1.5) = (2.2320.., 2, 1.5): cells (2,2,1), f = (2 r3 - 1.5, 0, .5)
    fx = 2 * r3 - 1.5
    jv = 0.5 * ((1 - fx) * (J[2, 2, 1] + J[2, 2, 2]) + fx * (J[3, 2, 1] + J[3, 2, 2]))
    I3 = I2 * exp(-K[2, 2, 1]) + jv * exp(-t2)
    t3 = t2 + K[2, 2, 1]
    for z in (1, 2):
        dep[2, 2, z] += 0.5 * (1 - fx) * I3
        dep[3, 2, z] += 0.5 * fx * I3
    # k=3: p = (0.5 + 3 r3, 2, 2.0) = (3.0980.., 2, 2): cell x = 3 (upper index clamps to 3), z cell 2 f = 0
    jv = J[3, 2, 2]
    I4 = I3 * exp(-K[3, 2, 2]) + jv * exp(-t3)
    dep[3, 2, 2] += I4
    j4, k4 = _grid4()
    tr = oracle_mod.trace_ray(j4[..., None], k4[..., None], (0.5, 2.0, 0.5), 0, 2, 1.0, 4, deposit=True)
    assert np.allclose(tr["I"][:, 0], [I1, I2, I3, I4], rtol=1e-13, atol=0)
    assert np.allclose(tr["acc"][..., 0], dep, rtol=1e-13, atol=1e-300)


def test_p6_negative_direction_clamps_at_zero(oracle_mod):
    # ray 1 of N_Omega = 2 has z = -1/2: it leaves through the low faces.  Uniform j, kappa make the
    # intensities closed-form (P1); the check is WHERE the mass lands once the ray is outside.
    nhat = oracle_mod.direction(1, 2)
    assert nhat[0] < 0 and nhat[1] > 0 and nhat[2] == -0.5
    j, kap = W.uniform_medium(4, 1.0, 0.0)
    tr = oracle_mod.trace_ray(j, kap, (0.25, 3.5, 0.25), 1, 2, 1.0, 6, deposit=True)
    # k=0 at (0.25, 3.5, 0.25): x cells {0,1}, y {3,3}, z {0,1}; from k=1 on x<0, y>3, z<0: everything on (0,3,0)
    assert np.all(tr["pos"][1:, 0] < 0) and np.all(tr["pos"][1:, 1] > 3) and np.all(tr["pos"][1:, 2] < 0)
    expect = np.zeros((4, 4, 4))
    I = np.arange(1, 7, dtype=np.float64)                      # kappa = 0, j = 1, ds = 1: I_k = k
    for x, wx in ((0, 0.75), (1, 0.25)):
        for z, wz in ((0, 0.75), (1, 0.25)):
            expect[x, 3, z] += wx * wz * I[0]
    expect[0, 3, 0] += I[1:].sum()
    assert np.allclose(tr["acc"][..., 0], expect, rtol=1e-14, atol=0)


# ------------------------------------------------------------------------------------------------------
# brute force on tiny NON-CUBIC grids: dense tent-function form of clamped trilinear read / deposit,
# position by the recurrence x_{k+1} = x_k + nhat ds (eq. 2 literally), clamping the POSITION (D5).
# ------------------------------------------------------------------------------------------------------
def _dense_reference(j, kap, src, nhats, ds, n_sub):
    shape = j.shape[:3]
    nb = j.shape[3]
    grids = np.meshgrid(*[np.arange(s, dtype=np.float64) for s in shape], indexing="ij")
    acc = np.zeros(j.shape)
    for nh in nhats:
        x = np.array(src, dtype=np.float64)
        I = np.zeros(nb)
        tau = np.zeros(nb)
        for _ in range(n_sub):
            xc = np.clip(x, 0.0, np.array(shape) - 1.0)
            tent = np.ones(shape)
            for a in range(3):
                tent = tent * np.maximum(0.0, 1.0 - np.abs(grids[a] - xc[a]))
            cell = tuple(np.minimum(np.floor(xc).astype(int), np.array(shape) - 1))
            kv = kap[cell].astype(np.float64)
            jv = np.tensordot(tent, j.astype(np.float64), axes=3)
            I = I * np.exp(-kv * ds) + jv * np.exp(-tau) * ds
            tau = tau + kv * ds
            acc += tent[..., None] * I
            x = x + nh * ds
    return acc * (FOUR_PI / len(nhats))


@pytest.mark.parametrize("shape,src", [((5, 4, 3), (2.3, 1.6, 0.8)), ((3, 6, 4), (0.0, 5.0, 1.5)),
                                        ((4, 4, 7), (-1.25, 1.5, 8.0))])
def test_brute_force_dense_tent_reference(oracle_mod, shape, src):
    rng = np.random.default_rng(sum(shape))
    j = rng.uniform(0.0, 2.0, shape + (2,)).astype(np.float32)
    kap = rng.uniform(0.0, 1.0, shape + (2,)).astype(np.float32)
    n_rays, ds, n_sub = 7, 0.4375, 12                                   # ds exact in binary: recurrence == closed form
    nhats = [oracle_mod.direction(i, n_rays) for i in range(n_rays)]
    ref = _dense_reference(j, kap, np.float32(src), nhats, ds, n_sub)
    out = oracle_mod.march(j, kap, np.array([src], np.float32), n_rays, ds, 1.0, ds * n_sub, 1)[0]
    assert np.allclose(out, ref, rtol=1e-11, atol=1e-14)


# ------------------------------------------------------------------------------------------------------
# P7  prefix property (reading D7): snapshot m of an n-step run == a 1-step run with dt' = (m+1) dt
# ------------------------------------------------------------------------------------------------------
def test_p7_snapshots_are_prefixes(oracle_mod):
    n = 24
    rho = W.lognormal_density(n, 21, 1.0)
    j = (1e-3 * rho ** 2)[..., None].astype(np.float32)
    kap = (0.05 * rho)[..., None].astype(np.float32)
    src = np.array([[5.5, 12.0, 17.25], [20.0, 3.0, 9.0]], np.float32)
    multi = oracle_mod.march(j, kap, src, 128, 0.5, 1.0, 3.0, 4, n_threads=1)
    for m in range(4):
        single = oracle_mod.march(j, kap, src, 128, 0.5, 1.0, 3.0 * (m + 1), 1, n_threads=1)
        assert np.allclose(multi[m], single[0], rtol=1e-13, atol=0)


# ------------------------------------------------------------------------------------------------------
# P8  optically thin limit (north_star): kappa = 0  =>  I_k = sum_{i<k} j(x_i) ds, with j(x_i) the clamped
#     trilinear read -- scipy.ndimage.map_coordinates(order=1, mode='nearest') is that read.
# ------------------------------------------------------------------------------------------------------
def test_p8_optically_thin_is_a_riemann_sum_of_trilinear_j(oracle_mod):
    from scipy.ndimage import map_coordinates
    rng = np.random.default_rng(8)
    shape = (9, 7, 8)
    jf = rng.uniform(0.0, 3.0, shape).astype(np.float32)
    j = jf[..., None]
    kap = np.zeros(shape + (1,), np.float32)
    src = np.float32([4.2, 3.3, 2.9])
    ds, n_sub, n_rays = 0.3, 30, 13
    for ray in range(n_rays):
        tr = oracle_mod.trace_ray(j, kap, src, ray, n_rays, ds, n_sub)
        nh = oracle_mod.direction(ray, n_rays)
        pos = src.astype(np.float64)[None, :] + (np.arange(n_sub) * f32(ds))[:, None] * nh[None, :]
        assert np.allclose(tr["pos"], pos, rtol=0, atol=1e-13)
        jv = map_coordinates(jf.astype(np.float64), pos.T, order=1, mode="nearest")
        assert np.allclose(tr["I"][:, 0], np.cumsum(jv) * f32(ds), rtol=1e-12, atol=0)
        assert np.all(tr["tau"] == 0.0)


# ------------------------------------------------------------------------------------------------------
# P9  linearity in j, additivity over sources, bins are independent problems
# ------------------------------------------------------------------------------------------------------
def test_p9_linearity_additivity_bins(oracle_mod):
    n = 20
    rho = W.lognormal_density(n, 9, 1.0)
    ks, js = W.bin_scalings(3)
    j = (1e-3 * rho ** 2)[..., None] * js
    kap = (0.05 * rho)[..., None] * ks
    j, kap = j.astype(np.float32), kap.astype(np.float32)
    src = np.array([[3.0, 4.5, 10.0], [15.5, 15.5, 2.0], [9.9, 0.1, 19.0]], np.float32)
    args = (64, 0.5, 1.0, 6.0, 2)
    full = oracle_mod.march(j, kap, src, *args, n_threads=1)
    # additivity over sources
    parts = sum(oracle_mod.march(j, kap, src[i:i + 1], *args, n_threads=1) for i in range(3))
    assert np.allclose(full, parts, rtol=1e-12, atol=1e-300)
    # a 3-bin run equals three 1-bin runs, bit for bit
    for b in range(3):
        one = oracle_mod.march(np.ascontiguousarray(j[..., b:b + 1]), np.ascontiguousarray(kap[..., b:b + 1]), src,
                               *args, n_threads=1)
        assert np.array_equal(one[..., 0], full[..., b])
    # linear in j (exact for a power of two)
    assert np.array_equal(oracle_mod.march(4 * j, kap, src, *args, n_threads=1), 4 * full)
    # thread count only changes the summation order
    assert np.allclose(oracle_mod.march(j, kap, src, *args, n_threads=3), full, rtol=1e-12, atol=1e-300)


# ------------------------------------------------------------------------------------------------------
# P10 trilinear consistency: j linear in the coordinates is read exactly inside the box; whole-cell
#     translations of source and fields translate the result
# ------------------------------------------------------------------------------------------------------
def test_p10_linear_field_and_translation(oracle_mod):
    n = 24
    a, b, c = np.meshgrid(*[np.arange(n, dtype=np.float64)] * 3, indexing="ij")
    al, be = np.array([0.5, 0.25, 0.125]), 2.0
    j = (be + al[0] * a + al[1] * b + al[2] * c)[..., None].astype(np.float32)      # exact in fp32
    kap = np.zeros((n, n, n, 1), np.float32)
    src = np.float32([11.5, 12.25, 10.75])
    ds, n_sub = 0.5, 16                                                            # stays inside the box
    for ray in (0, 5, 22):
        nh = oracle_mod.direction(ray, 23)
        tr = oracle_mod.trace_ray(j, kap, src, ray, 23, ds, n_sub)
        k = np.arange(1, n_sub + 1)
        # I_k = ds * sum_{i<k} [be + al.(x0 + i ds nhat)] = ds [k (be + al.x0) + ds (al.nhat) k(k-1)/2]
        expect = ds * (k * (be + al @ src.astype(np.float64)) + ds * (al @ nh) * k * (k - 1) / 2)
        assert np.allclose(tr["I"][:, 0], expect, rtol=1e-13, atol=0)
    # translation by whole cells, far from the walls (horizon 4 < distance to any wall)
    rho = W.lognormal_density(n, 4, 1.0)
    jj = (1e-3 * rho ** 2)[..., None].astype(np.float32)
    kk = (0.05 * rho)[..., None].astype(np.float32)
    s0 = np.array([[9.3, 10.1, 8.6]], np.float32)
    shift = (3, 2, 5)
    base = oracle_mod.march(jj, kk, s0, 48, 0.5, 1.0, 4.0, 1)[0]
    moved = oracle_mod.march(np.roll(jj, shift, (0, 1, 2)), np.roll(kk, shift, (0, 1, 2)),
                             s0 + np.float32(shift), 48, 0.5, 1.0, 4.0, 1)[0]
    assert np.allclose(np.roll(base, shift, (0, 1, 2)), moved, rtol=1e-9, atol=1e-300)
    assert base.sum() > 0


def test_config_c0_matches_its_recipe(oracle_mod):
    """C0 (BASELINE.json configs[0]) end to end: mass from per-ray traces and the horizon."""
    w = W.make_config("C0")
    out = oracle_mod.march(w.j, w.kappa, w.sources, w.n_rays, w.step_size, w.c, w.dt, w.n_steps)
    assert out.shape == (1, 16, 16, 16, 1)
    mass = sum(oracle_mod.trace_ray(w.j, w.kappa, w.sources[0], i, w.n_rays, w.step_size, 24)["I"].sum()
               for i in range(w.n_rays))
    assert out.sum() == pytest.approx(FOUR_PI / w.n_rays * mass, rel=1e-12)
    assert oracle_mod.substeps(w.step_size, w.c, w.dt) == w.substeps_per_step == 24


# ------------------------------------------------------------------------------------------------------
# D17  stepping with explicit ray state (oracle.step; "fix dt and iterate")
# ------------------------------------------------------------------------------------------------------
def test_d17_steps_in_a_static_medium_add_up_to_the_snapshots(oracle_mod):
    rho = W.lognormal_density(12, 5, 1.0)
    ks, js = W.bin_scalings(3)
    j = np.ascontiguousarray((1e-2 * rho ** 2)[..., None] * js, dtype=np.float32)
    kap = np.ascontiguousarray((0.1 * rho)[..., None] * ks, dtype=np.float32)
    src = np.array([[5.5, 6.0, 3.25], [-1.0, 4.0, 13.5]], dtype=np.float32)
    n_rays, ds, dt, n_steps = 37, 0.5, 3.0, 4
    snaps = oracle_mod.march(j, kap, src, n_rays, ds, 1.0, dt, n_steps)
    state = oracle_mod.new_state(2, n_rays, 3)
    ns = oracle_mod.substeps(ds, 1.0, dt)
    run = np.zeros_like(snaps[0])
    for m in range(n_steps):
        run += oracle_mod.step(j, kap, src, n_rays, ds, 1.0, dt, m * ns, state)
        assert np.abs(run - snaps[m]).max() <= 1e-12 * snaps[m].max()
    assert (state[:, :, 1, :] > 0).all()          # tau grew on every ray


def test_d17_medium_changed_between_steps_closed_form(oracle_mod):
    """Uniform (j1, k1) during step 1, uniform (j2, k2) during step 2: by induction on eq. (2)
    I_{N+i} = I_N a2^i + i j2 ds e^{-tau_N} a2^{i-1}, with I_N = N j1 ds a1^{N-1}, tau_N = N k1 ds."""
    n, n_rays, ds, dt = 10, 24, 0.5, 3.0
    N = oracle_mod.substeps(ds, 1.0, dt)
    j1, k1, j2, k2 = f32(0.3), f32(0.2), f32(0.7), f32(0.05)
    src = np.array([[4.5, 4.5, 4.5], [8.0, 1.0, 2.0]], dtype=np.float32)
    state = oracle_mod.new_state(2, n_rays, 1)
    ja, ka = W.uniform_medium(n, j1, k1)
    jb, kb = W.uniform_medium(n, j2, k2)
    oracle_mod.step(ja, ka, src, n_rays, ds, 1.0, dt, 0, state)
    a1, a2 = math.exp(-k1 * ds), math.exp(-k2 * ds)
    I_N, tau_N = N * j1 * ds * a1 ** (N - 1), N * k1 * ds
    assert np.allclose(state[:, :, 0, 0], I_N, rtol=1e-13) and np.allclose(state[:, :, 1, 0], tau_N, rtol=1e-13)
    inc = oracle_mod.step(jb, kb, src, n_rays, ds, 1.0, dt, N, state)
    I_end = I_N * a2 ** N + N * j2 * ds * math.exp(-tau_N) * a2 ** (N - 1)
    assert np.allclose(state[:, :, 0, 0], I_end, rtol=1e-13)
    assert np.allclose(state[:, :, 1, 0], tau_N + N * k2 * ds, rtol=1e-13)
    mass = sum(I_N * a2 ** i + i * j2 * ds * math.exp(-tau_N) * a2 ** (i - 1) for i in range(1, N + 1))
    assert abs(inc.sum() - FOUR_PI * 2 * mass) <= 1e-12 * inc.sum()      # every substep deposits total weight 1


def test_d17_a_step_sees_only_its_own_medium(oracle_mod):
    """j = 0 in step 2 with kappa = 0: the intensity of step 1 is carried unchanged and keeps being deposited;
    positions continue the same straight line (the increment equals a static-medium run's, scaled)."""
    n, n_rays, ds, dt = 8, 16, 0.5, 2.0
    N = oracle_mod.substeps(ds, 1.0, dt)
    ja, ka = W.uniform_medium(n, 0.4, 0.0)
    jz, kz = W.uniform_medium(n, 0.0, 0.0)
    src = np.array([[3.5, 3.5, 3.5]], dtype=np.float32)
    state = oracle_mod.new_state(1, n_rays, 1)
    oracle_mod.step(ja, ka, src, n_rays, ds, 1.0, dt, 0, state)
    I_N = N * f32(0.4) * ds
    inc = oracle_mod.step(jz, kz, src, n_rays, ds, 1.0, dt, N, state)
    assert np.allclose(state[:, :, 0, 0], I_N, rtol=1e-14)
    # the same geometry deposited with unit intensity: a static run with I forced to 1 does not exist, but the
    # deposit pattern of substeps N..2N-1 is that of (snapshot 2 - snapshot 1) of a run whose I is constant:
    # j = 0, kappa = 0 after an initial state of I = 1 <=> linearity in the carried intensity
    state1 = oracle_mod.new_state(1, n_rays, 1)
    state1[:, :, 0, 0] = 1.0
    unit = oracle_mod.step(jz, kz, src, n_rays, ds, 1.0, dt, N, state1)
    assert np.abs(inc - I_N * unit).max() <= 1e-13 * inc.max()
    assert abs(unit.sum() - FOUR_PI * N) <= 1e-12 * unit.sum()


# ------------------------------------------------------------------------------------------------------
# D18  trilinear kappa variant (PAPER.md:29 samples kappa nearest-neighbour "(currently)")
# ------------------------------------------------------------------------------------------------------
def test_d18_uniform_kappa_cannot_tell_the_readings_apart(oracle_mod):
    rho = W.lognormal_density(10, 9, 1.0)
    j = np.ascontiguousarray((1e-2 * rho ** 2)[..., None], dtype=np.float32)
    kap = np.full(j.shape, 0.15, dtype=np.float32)
    src = np.array([[4.4, 5.1, 3.3]], dtype=np.float32)
    a = oracle_mod.march(j, kap, src, 50, 0.5, 1.0, 6.0, 2)
    b = oracle_mod.march(j, kap, src, 50, 0.5, 1.0, 6.0, 2, kappa_trilinear=True)
    assert np.abs(a - b).max() <= 1e-13 * a.max()


def test_d18_tau_is_the_riemann_sum_of_the_library_trilinear_read(oracle_mod):
    """tau_k = ds * sum_{i<k} kappa(x_i) with kappa read by scipy's order-1 map_coordinates, mode 'nearest'
    (= clamped indices), along rays that leave the box."""
    from scipy.ndimage import map_coordinates
    rng = np.random.default_rng(21)
    shape = (7, 6, 5)
    kap = rng.uniform(0.0, 0.6, shape + (2,)).astype(np.float32)
    j = rng.uniform(0.1, 1.0, shape + (2,)).astype(np.float32)
    src, ds, n_sub = (3.3, 2.6, 1.9), 0.37, 30
    for ray in (0, 5, 11, 22):
        tr = oracle_mod.trace_ray(j, kap, src, ray, 23, ds, n_sub, kappa_trilinear=True)
        for b in range(2):
            kx = map_coordinates(kap[..., b].astype(np.float64), tr["pos"].T, order=1, mode="nearest")
            assert np.abs(tr["tau"][:, b] - f32(ds) * np.cumsum(kx)).max() <= 1e-12
        nn = oracle_mod.trace_ray(j, kap, src, ray, 23, ds, n_sub)
        assert np.abs(nn["tau"] - tr["tau"]).max() > 1e-3          # and it is a different reading from D4


def test_d18_hand_trace_axis_ray(oracle_mod):
    """N_Omega = 1 (nhat = (1,0,0)), source on a node: x-fractions alternate 0 and 1/2, so kappa is a cell value
    or the mean of two neighbours; after the box, the boundary value (clamped)."""
    J, K = _grid4()
    J, K = J.astype(np.float64), K.astype(np.float64)
    ds, y, z = 0.5, 1, 2
    I = tau = 0.0
    want = []
    for k in range(10):
        x = 1.0 + k * ds
        i0, f = int(math.floor(x)), x - math.floor(x)
        lo, hi = min(i0, 3), min(i0 + 1, 3)
        kap = (1 - f) * K[lo, y, z] + f * K[hi, y, z]
        jv = (1 - f) * J[lo, y, z] + f * J[hi, y, z]
        I = I * math.exp(-kap * ds) + jv * math.exp(-tau) * ds
        tau += kap * ds
        want.append((I, tau))
    j4, k4 = _grid4()
    tr = oracle_mod.trace_ray(j4[..., None], k4[..., None], (1.0, 1.0, 2.0), 0, 1, ds, 10, kappa_trilinear=True)
    assert np.allclose(tr["I"][:, 0], [w[0] for w in want], rtol=1e-14)
    assert np.allclose(tr["tau"][:, 0], [w[1] for w in want], rtol=1e-14)


# ------------------------------------------------------------------------------------------------------
# D19  adjoint of the march with respect to j.  The forward oracle is pinned above; the adjoint
#      is pinned against it by the identity that DEFINES a transpose, <A j, g> = <j, A^T g>, for random j and g.
# ------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("shape,nb,n_src,n_rays,ds,dt,n_steps", [
    ((6, 5, 7), 1, 2, 13, 0.5, 4.0, 1),
    ((5, 4, 3), 3, 3, 7, 0.37, 2.6, 3),         # several snapshots: gbar[m] acts on the CUMULATIVE field of step m
    ((4, 4, 4), 2, 1, 1, 0.5, 5.0, 2),          # the axis ray, leaving the box (clamped deposits)
])
def test_d19_adjoint_is_the_transpose_of_the_march(oracle_mod, shape, nb, n_src, n_rays, ds, dt, n_steps):
    rng = np.random.default_rng(sum(shape) + nb)
    kap = rng.uniform(0.0, 0.6, shape + (nb,)).astype(np.float32)
    src = rng.uniform(-1.0, max(shape), (n_src, 3)).astype(np.float32)
    for trial in range(3):
        j = rng.uniform(-1.0, 1.0, shape + (nb,)).astype(np.float32)           # signs allowed: the map is linear
        g = rng.standard_normal((n_steps,) + shape + (nb,))
        out = oracle_mod.march(j, kap, src, n_rays, ds, 1.0, dt, n_steps)
        grad = oracle_mod.adjoint_j(g, kap, src, n_rays, ds, 1.0, dt, n_steps)
        lhs, rhs = float((out * g).sum()), float((j.astype(np.float64) * grad).sum())
        assert abs(lhs - rhs) <= 1e-11 * max(np.abs(out * g).sum(), 1e-300), (lhs, rhs)


def test_d19_column_of_the_operator(oracle_mod):
    """grad_j for gbar = a unit impulse at voxel v is row v of A: it equals the response at v to unit emissivity
    placed voxel by voxel (brute force over all 27 cells of a 3^3 grid)."""
    shape, n_rays, ds, dt = (3, 3, 3), 6, 0.5, 2.0
    rng = np.random.default_rng(3)
    kap = rng.uniform(0.1, 0.5, shape + (1,)).astype(np.float32)
    src = np.array([[1.2, 0.9, 1.4]], dtype=np.float32)
    v = (2, 1, 0, 0)
    g = np.zeros((1,) + shape + (1,))
    g[(0,) + v] = 1.0
    grad = oracle_mod.adjoint_j(g, kap, src, n_rays, ds, 1.0, dt, 1)
    for cell in np.ndindex(*shape):
        j = np.zeros(shape + (1,), dtype=np.float32)
        j[cell + (0,)] = 1.0
        resp = oracle_mod.march(j, kap, src, n_rays, ds, 1.0, dt, 1)[(0,) + v]
        assert abs(resp - grad[cell + (0,)]) <= 1e-13 * max(abs(resp), 1e-30)


def test_d19_scalar_amplitude_inversion_matches_the_closed_form(oracle_mod):
    """The paper's demo: recover A in j = A e0 from I_ref by minimising the MSE.  The loss is a parabola in A;
    gradient descent with dL/dA = <e0, A^T (2/n)(A_op(A e0) - I_ref)> reaches the closed-form minimiser
    <F, I_ref>/<F, F>, F = A_op e0."""
    n = 8
    rho = W.lognormal_density(n, 4, 0.8)
    e0 = np.ascontiguousarray((rho ** 2)[..., None], dtype=np.float32)
    kap = np.ascontiguousarray((0.1 * rho)[..., None], dtype=np.float32)
    src = np.array([[3.5, 3.5, 3.5]], dtype=np.float32)
    args = (src, 24, 0.5, 1.0, 3.0, 1)
    F = oracle_mod.march(e0, kap, *args)
    A_true = 2.5
    I_ref = A_true * F + 0.01 * F.max() * np.random.default_rng(0).standard_normal(F.shape)
    A_star = float((F * I_ref).sum() / (F * F).sum())
    A = 0.3
    lip = 2.0 * float((F * F).sum()) / F.size
    for _ in range(40):
        resid = A * F - I_ref
        dLdA = float((e0.astype(np.float64) * oracle_mod.adjoint_j(2.0 * resid / F.size, kap, *args)).sum())
        assert abs(dLdA - 2.0 * float((resid * F).sum()) / F.size) <= 1e-11 * 2.0 * float(np.abs(resid * F).sum()) / F.size
        A -= dLdA / lip
    assert abs(A - A_star) <= 1e-9 * abs(A_star)


def test_d20_relative_mse_inversion_matches_its_closed_form(oracle_mod):
    """The paper's other loss ("either a plain MSE or a relative MSE"; reading D20): L(A) = mean(w (A F - I_ref)^2),
    w = 1 / (I_ref^2 + eps^2).  Still a parabola in A: gradient descent with dL/dA = <e0, A^T (2/n) w (A F - I_ref)>
    reaches <w F, I_ref> / <w F, F> ("the corresponding closed-form minimizer (under the chosen weighting)"), which
    differs from the plain-MSE minimiser."""
    n = 8
    rho = W.lognormal_density(n, 4, 0.8)
    e0 = np.ascontiguousarray((rho ** 2)[..., None], dtype=np.float32)
    kap = np.ascontiguousarray((0.1 * rho)[..., None], dtype=np.float32)
    src = np.array([[3.5, 3.5, 3.5]], dtype=np.float32)
    args = (src, 24, 0.5, 1.0, 3.0, 1)
    F = oracle_mod.march(e0, kap, *args)
    I_ref = 2.5 * F * (1.0 + 0.1 * np.random.default_rng(0).standard_normal(F.shape))
    eps = 1e-3 * I_ref.max()
    wgt = 1.0 / (I_ref ** 2 + eps ** 2)
    A_star = float((wgt * F * I_ref).sum() / (wgt * F * F).sum())
    lip = 2.0 * float((wgt * F * F).sum()) / F.size
    A = 0.3
    for _ in range(40):
        resid = A * F - I_ref
        dLdA = float((e0.astype(np.float64) * oracle_mod.adjoint_j(2.0 * wgt * resid / F.size, kap, *args)).sum())
        A -= dLdA / lip
    assert abs(A - A_star) <= 1e-9 * abs(A_star)
    assert abs(float((F * I_ref).sum() / (F * F).sum()) - A_star) > 1e-3 * abs(A_star)


# ------------------------------------------------------------------------------------------------------
# D19  adjoint with respect to kappa: pinned by central differences of the (pinned) forward oracle
# ------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("shape,nb,n_src,n_rays,ds,dt,n_steps", [
    ((5, 4, 6), 1, 2, 9, 0.5, 4.0, 1),
    ((4, 5, 3), 2, 1, 7, 0.37, 2.6, 3),          # snapshots are cumulative: earlier substeps feed every later gbar[m]
    ((4, 4, 4), 1, 1, 1, 0.5, 5.0, 2),           # axis ray leaving the box
])
def test_d19_kappa_gradient_matches_central_differences(oracle_mod, shape, nb, n_src, n_rays, ds, dt, n_steps):
    rng = np.random.default_rng(sum(shape) * 7 + nb)
    kap = rng.uniform(0.05, 0.6, shape + (nb,))
    j = rng.uniform(0.1, 1.0, shape + (nb,)).astype(np.float32)
    src = rng.uniform(0.0, min(shape) - 1.0, (n_src, 3)).astype(np.float32)
    g = rng.standard_normal((n_steps,) + shape + (nb,))
    # kappa values exactly representable in fp32 with room for the perturbation (the oracle reads fp32 arrays)
    kap = np.round(kap * 1024) / 1024
    grad = oracle_mod.adjoint_kappa(g, j, kap.astype(np.float32), src, n_rays, ds, 1.0, dt, n_steps)

    def loss(k):
        return float((oracle_mod.march(j, k.astype(np.float32), src, n_rays, ds, 1.0, dt, n_steps) * g).sum())

    eps = 2.0 ** -12
    for trial in range(4):                                    # directional derivatives
        d = np.round(rng.uniform(-1.0, 1.0, kap.shape) * 16) / 16
        fd = (loss(kap + eps * d) - loss(kap - eps * d)) / (2 * eps)
        an = float((grad * d).sum())
        assert abs(fd - an) <= 5e-6 * max(abs(an), np.abs(grad * d).sum() * 1e-3), (fd, an)
    for cell in [tuple(rng.integers(0, n) for n in shape) + (0,) for _ in range(3)]:   # single entries
        e = np.zeros_like(kap)
        e[cell] = 1.0
        fd = (loss(kap + eps * e) - loss(kap - eps * e)) / (2 * eps)
        assert abs(fd - grad[cell]) <= 5e-6 * max(abs(grad[cell]), np.abs(grad).max() * 1e-3), (cell, fd, grad[cell])


def test_d19_kappa_gradient_uniform_medium_closed_form(oracle_mod):
    """Uniform j0, kappa0: I_{k+1} = (k+1) j0 ds a^k, so with gbar = 1 everywhere (L = total deposited field)
    dL/dkappa0 = sum over voxels of grad_kappa = 4 pi n_src d/dkappa0 [sum_k (k+1) j0 ds a^k]."""
    n, n_rays, ds, dt = 8, 12, 0.5, 5.0
    N = oracle_mod.substeps(ds, 1.0, dt)
    j0, k0 = f32(0.3), f32(0.25)
    j, kap = W.uniform_medium(n, j0, k0)
    src = np.array([[3.5, 3.5, 3.5], [1.0, 6.0, 2.5]], dtype=np.float32)
    g = np.ones((1, n, n, n, 1))
    grad = oracle_mod.adjoint_kappa(g, j, kap, src, n_rays, ds, 1.0, dt, 1)
    a = math.exp(-k0 * ds)
    want = FOUR_PI * 2 * sum((k + 1) * j0 * ds * k * (-ds) * a ** k for k in range(N))
    assert abs(grad.sum() - want) <= 1e-12 * abs(want)


# ------------------------------------------------------------------------------------------------------
# D21  forward-mode derivative with respect to kappa: pinned by central differences of the (pinned) forward
#      oracle, by its duality with the (pinned) kappa adjoint, and by a uniform-medium closed form
# ------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("shape,nb,n_src,n_rays,ds,dt,n_steps", [
    ((5, 4, 6), 1, 2, 9, 0.5, 4.0, 1),
    ((4, 5, 3), 2, 1, 7, 0.37, 2.6, 3),          # several cumulative snapshots
    ((4, 4, 4), 1, 1, 1, 0.5, 5.0, 2),           # axis ray leaving the box (clamped deposits go on)
])
def test_d21_jvp_kappa_matches_central_differences_and_the_adjoint(oracle_mod, shape, nb, n_src, n_rays, ds, dt, n_steps):
    rng = np.random.default_rng(sum(shape) * 11 + nb)
    kap = np.round(rng.uniform(0.05, 0.6, shape + (nb,)) * 1024) / 1024        # exactly representable with room for eps
    j = rng.uniform(0.1, 1.0, shape + (nb,)).astype(np.float32)
    src = rng.uniform(0.0, min(shape) - 1.0, (n_src, 3)).astype(np.float32)
    args = (src, n_rays, ds, 1.0, dt, n_steps)
    eps = 2.0 ** -12
    for trial in range(3):
        d = np.round(rng.uniform(-1.0, 1.0, kap.shape) * 16) / 16
        tang = oracle_mod.jvp_kappa(j, kap.astype(np.float32), d.astype(np.float32), *args)
        fd = (oracle_mod.march(j, (kap + eps * d).astype(np.float32), *args) -
              oracle_mod.march(j, (kap - eps * d).astype(np.float32), *args)) / (2 * eps)
        assert np.abs(tang - fd).max() <= 2e-6 * np.abs(fd).max(), np.abs(tang - fd).max() / np.abs(fd).max()
        # duality: <g, J d> = <J^T g, d> with J^T g from the kappa adjoint (pinned on its own above)
        g = rng.standard_normal(tang.shape)
        lhs = float((g * tang).sum())
        rhs = float((oracle_mod.adjoint_kappa(g, j, kap.astype(np.float32), *args) * d).sum())
        assert abs(lhs - rhs) <= 1e-11 * max(abs(lhs), np.abs(g * tang).sum() * 1e-3), (lhs, rhs)


def test_d21_global_kappa_scale_uniform_medium_closed_form(oracle_mod):
    """The paper's example of a further parameter ("a global kappa scale"): kappa = theta kappa0, uniform j0.  Every
    ray has I_k = k j0 ds a^(k-1), a = exp(-theta kappa0 ds) (pin P1), every substep deposits total weight 1 (P2), so
    sum(out) = 4 pi n_src j0 ds sum_{k=1..N} k a^(k-1) and
    d/dtheta sum(out) = 4 pi n_src j0 ds sum_k k (k-1) a^(k-2) (-kappa0 ds a); the tangent for dkappa = kappa sums to it."""
    n, j0, k0, ds, N = 9, 0.3, 0.2, 0.5, 14
    j = np.full((n, n, n, 1), j0, dtype=np.float32)
    kap = np.full((n, n, n, 1), k0, dtype=np.float32)
    src = np.array([[4.0, 4.0, 4.0], [1.5, 6.25, 3.0]], dtype=np.float32)
    tang = oracle_mod.jvp_kappa(j, kap, kap, src, 24, ds, 1.0, N * ds, 1)
    a = np.exp(-float(np.float32(k0)) * ds)
    j0f, k0f = float(np.float32(j0)), float(np.float32(k0))
    want = 4 * np.pi * len(src) * j0f * ds * sum(k * (k - 1) * a ** (k - 2) for k in range(1, N + 1)) * (-k0f * ds * a)
    assert abs(tang.sum() - want) <= 1e-12 * abs(want), (tang.sum(), want)
    assert (tang <= 0).all()                      # more absorption, less field, everywhere
