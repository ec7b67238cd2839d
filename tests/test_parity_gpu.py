"""GPU-vs-oracle parity (tier T2/T3): every test calls the CUDA path through the C ABI (ctypes binding) and
compares with the fp64 oracle on the same seeded inputs, element by element, at BASELINE.json's tolerances
(relative L2 <= 1e-4; per-voxel relative error <= 1e-3 on voxels above 1e-6 of the field maximum).

Sizes: C0 and C1 in full; C2/C3/C4 against the oracle on stratified SOURCE SUBSETS (the field is a plain sum
over sources, so a subset is the same computation with fewer terms; every other argument is the
config's own), and at FULL size — the launch configuration bench.py times — through properties that hold at
any size: additivity over source chunks, exact darkness beyond the light front, run-to-run agreement, the
prefix property — and against the oracle on the WHOLE config (test_full_size_oracle_parity; the fp64 oracle
needs tens of seconds per config on the GPU box's host cores; RT_SKIP_FULL_PARITY=1 skips it).
"""
import os

import numpy as np
import pytest

import parity
import workloads

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def rt():
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device")
    import paper_2511_09389_b200 as rt
    return rt


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def gpu_march(rt, w, variant=0, sources=None, n_steps=None, dt=None):
    src = w.sources if sources is None else sources
    out = rt.rt_march_ex(_dev(w.j), _dev(w.kappa), _dev(src), w.n_rays, w.step_size, w.c,
                         w.dt if dt is None else dt, w.n_steps if n_steps is None else n_steps, variant=variant)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def oracle_march(oracle_mod, w, sources=None):
    src = w.sources if sources is None else sources
    return oracle_mod.march(w.j, w.kappa, src, w.n_rays, w.step_size, w.c, w.dt, w.n_steps)


_cache = {}


def config(name):
    if name not in _cache:
        _cache.clear()              # one large config in memory at a time
        _cache[name] = workloads.make_config(name)
    return _cache[name]


def _stratified(n_src, count):
    return np.unique(np.linspace(0, n_src - 1, count).round().astype(int))


VARIANTS = [0, 1, 2, 3, 4, 5, 16, 17, 21, 32, 36, 53]   # kinds 0..5; flags: 16 fp32 accumulation, 32 one bin per thread


# ------------------------------------------------------------------------------------------------
# building blocks
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [1, 2, 5, 7, 33, 40, 64, 1000, 4096, 16384])
def test_directions_match_oracle(rt, oracle_mod, n):
    got = rt.rt_directions(n).cpu().numpy()
    want = np.stack([oracle_mod.direction(i, n) for i in range(n)])
    # z and the radius are stated as correctly rounded IEEE operations on both sides (D1/D3): z is
    # bit-identical; x, y differ only by the two libraries' sin/cos of the azimuth (a few ulp of 1)
    assert np.array_equal(got[:, 2], want[:, 2])
    assert np.abs(got - want).max() <= 1e-15
    if n == 1:
        assert got[0].tolist() == [1.0, 0.0, 0.0]          # the hand-traceable axis ray (pin P6)
    if n == 5:
        assert got[0, 0] == want[0, 0] and got[0, 1] == 0.0    # azimuth 0: x is the radius itself, same bits


@pytest.mark.parametrize("shape,nb,src,n_rays,ds,n_sub", [
    ((5, 4, 3), 3, (0.0, 3.0, 2.0), 7, 0.5, 10),            # rays whose z-position lands exactly on integer planes
    ((3, 6, 4), 4, (0.0, 5.0, 1.5), 33, 0.25, 12),
    ((6, 5, 7), 8, (-3.0, 9.0, 2.5), 40, 0.5, 48),
    ((6, 5, 7), 1, (1.0, 2.0, 0.0), 5, 0.5, 24),            # ray 0 is (0.6, 0, 0.8) up to rounding
    ((16, 16, 16), 2, (7.5, 7.25, 8.0), 64, 0.5, 40),
    ((8, 8, 8), 1, (3.5, 3.5, 3.5), 50, 1.7, 8),
])
def test_single_ray_traces_match_oracle(rt, oracle_mod, shape, nb, src, n_rays, ds, n_sub):
    """Per-substep parity of one ray: x_k (same 2^-64 grid point, so the same cell), I_{k+1}, exp(-tau_{k+1})."""
    j, k = _random_medium(shape, nb, seed=sum(shape) + nb)
    dj, dk, dsrc = _dev(j), _dev(k), _dev(np.array(src, dtype=np.float32))
    for ray in range(n_rays):
        g = rt.rt_trace_ray(dj, dk, dsrc, ray, n_rays, ds, n_sub)
        o = oracle_mod.trace_ray(j, k, src, ray, n_rays, ds, n_sub)
        gp = g["pos"].cpu().numpy()
        # z has the same bits on both sides => the same grid point on axis 2, in particular the same floor
        assert np.array_equal(np.floor(gp[:, 2]), np.floor(o["pos"][:, 2])), (ray, gp[:, 2], o["pos"][:, 2])
        assert np.abs(gp - o["pos"]).max() <= 2e-14 * max(1.0, np.abs(o["pos"]).max())
        gi, gt = g["I"].cpu().numpy().astype(np.float64), g["T"].cpu().numpy().astype(np.float64)
        assert np.abs(gi - o["I"]).max() <= 2e-5 * o["I"].max(), ray
        assert (np.abs(gt - np.exp(-o["tau"])) <= 2e-5 * np.exp(-o["tau"]) + 1e-37).all(), ray


@pytest.mark.parametrize("n", [1, 31, 64, 1000, 4096, 16384, 100003])
def test_ray_order_is_a_permutation(rt, n):
    order = rt.rt_ray_order(n).cpu().numpy().astype(np.int64) & 0xFFFFFFFF
    real = order[order != 0xFFFFFFFF]
    assert len(order) == rt.rt_ray_slots(n)
    assert np.array_equal(np.sort(real), np.arange(n))


def test_substeps_rule_matches_oracle(rt, oracle_mod):
    rng = np.random.default_rng(5)
    cases = [(0.5, 1.0, 12.0), (0.5, 1.0, 222.0), (0.1, 1.0, 0.3), (0.3, 2.0, 1.0), (1.0, 1.0, 1e-3), (0.7, 3.0, 9.1)]
    cases += [tuple(np.float32(rng.uniform(0.05, 3.0, 3))) for _ in range(200)]
    for ds, c, dt in cases:
        assert rt.rt_substeps_per_step(ds, c, dt) == oracle_mod.substeps(ds, c, dt), (ds, c, dt)


# ------------------------------------------------------------------------------------------------
# C0, C1: full configs, every kernel variant, every snapshot
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("name", ["C0", "C1"])
def test_small_configs_full_parity(rt, oracle_mod, name, variant):
    w = config(name)
    ref = oracle_march(oracle_mod, w)
    got = gpu_march(rt, w, variant)
    parity.assert_parity(got, ref, f"{name} variant {variant}")


def test_single_source_entry_point(rt, oracle_mod):
    w = config("C0")
    out = rt.rt_march_single(_dev(w.j), _dev(w.kappa), _dev(w.sources[0]), w.n_rays, w.step_size, w.c, w.dt,
                             w.n_steps)
    torch.cuda.synchronize()
    parity.assert_parity(out.cpu().numpy(), oracle_march(oracle_mod, w), "rt_march_single C0")


def test_host_entry_point(rt, oracle_mod):
    w = config("C1")
    out = rt.rt_march_host(w.j, w.kappa, w.sources, w.n_rays, w.step_size, w.c, w.dt, w.n_steps)
    parity.assert_parity(out, oracle_march(oracle_mod, w), "rt_march_host C1")


# ------------------------------------------------------------------------------------------------
# hand-traceable and degenerate cases
# ------------------------------------------------------------------------------------------------
def _random_medium(shape, nb, seed):
    rng = np.random.default_rng(seed)
    j = rng.uniform(0.1, 1.0, shape + (nb,)).astype(np.float32)
    k = rng.uniform(0.0, 0.6, shape + (nb,)).astype(np.float32)
    return j, k


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("shape,nb,src,n_rays,ds,dt", [
    ((4, 4, 4), 1, [(1.0, 2.0, 1.0)], 1, 0.5, 4.0),            # axis ray through and out of a 4-cube (pin P6)
    ((4, 4, 4), 1, [(2.0, 1.0, 2.0)], 2, 0.5, 4.0),            # N_Omega = 2
    ((5, 4, 3), 3, [(2.3, 1.6, 0.8), (0.0, 3.0, 2.0)], 7, 0.5, 5.0),   # ragged shape, 3 bins (scalar path)
    ((3, 6, 4), 4, [(0.0, 5.0, 1.5)], 33, 0.25, 3.0),          # 4 bins (v4 path), source on a face
    ((6, 5, 7), 8, [(-3.0, 9.0, 2.5)], 40, 0.5, 8.0),          # 8 bins, source OUTSIDE the box (clamped)
    ((1, 1, 1), 1, [(0.0, 0.0, 0.0)], 5, 0.5, 2.0),            # one-voxel grid: everything clamps to it
    ((2, 9, 1), 5, [(0.5, 4.0, 0.0)], 19, 0.5, 6.0),           # flat grid, 5 bins
    ((8, 8, 8), 1, [(3.5, 3.5, 3.5)], 50, 1.7, 13.6),          # steps longer than a cell (stencil jumps)
    ((8, 8, 8), 4, [(3.0, 4.0, 5.0)], 50, 0.05, 1.0),          # many substeps per cell
    ((8, 8, 8), 1, [(3.5, 3.5, 3.5)], 17, 0.5, 0.4),           # N_s = 1
])
def test_small_cases(rt, oracle_mod, shape, nb, src, n_rays, ds, dt, variant):
    j, k = _random_medium(shape, nb, seed=sum(shape) + nb)
    src = np.array(src, dtype=np.float32)
    for n_steps in (1, 3):
        ref = oracle_mod.march(j, k, src, n_rays, ds, 1.0, dt, n_steps)
        out = rt.rt_march_ex(_dev(j), _dev(k), _dev(src), n_rays, ds, 1.0, dt, n_steps, variant=variant)
        torch.cuda.synchronize()
        parity.assert_parity(out.cpu().numpy(), ref, f"{shape} nb={nb} variant={variant} steps={n_steps}")


@pytest.mark.parametrize("variant", [0, 4, 5, 21])
@pytest.mark.parametrize("n_src,integer", [(32, True), (33, False), (70, True), (100, False)])
def test_many_sources_fill_warps_raggedly(rt, oracle_mod, n_src, integer, variant):
    """n_src >= 32 selects the warp = 32 sorted sources x 1 direction mapping: ragged last source group,
    duplicate sources, sources on faces and outside the box (clamped), cell-centred and not."""
    shape, nb, n_rays = (7, 6, 9), 1, 11
    j, k = _random_medium(shape, nb, seed=n_src)
    rng = np.random.default_rng(1000 + n_src)
    src = rng.uniform(-2.0, 10.0, (n_src, 3))
    if integer:
        src = np.round(src)
    src[1] = src[0]                                   # a duplicate
    src[2] = (0.0, 5.0, 8.0)                          # on three faces
    src = src.astype(np.float32)
    ref = oracle_mod.march(j, k, src, n_rays, 0.5, 1.0, 4.0, 2)
    out = rt.rt_march_ex(_dev(j), _dev(k), _dev(src), n_rays, 0.5, 1.0, 4.0, 2, variant=variant)
    torch.cuda.synchronize()
    parity.assert_parity(out.cpu().numpy(), ref, f"n_src={n_src} variant={variant}")


@pytest.mark.parametrize("case", ["quarter_fractions", "one_source_off", "integer_outside", "long_steps", "two_warps",
                                  "tiny_negative_offsets"])
def test_sources_sharing_their_cell_fractions(rt, oracle_mod, case):
    """>= 32 sources, one bin: warp = 32 sorted sources x 1 direction.  Sources that share their fractional cell
    offsets (the lanes then cross cell planes in the same substep) with non-zero fractions, one source breaking the
    pattern, sources outside the box, substeps longer than a cell, a ragged last source group and exactly two full
    groups; reductions spread over the copies of the accumulation grid.  Against the oracle and against the
    textbook-order kernel variant."""
    shape, n_rays, ds, dt, n_steps = (9, 7, 8), 37, 0.25, 9.25, 3            # 37 substeps per step
    rng = np.random.default_rng(77)
    n_src = 45
    src = rng.integers(-1, 10, (n_src, 3)).astype(np.float64)
    if case == "quarter_fractions":
        src += (0.25, 0.5, 0.75)
    elif case == "one_source_off":
        src += (0.25, 0.5, 0.75)
        src[31, 1] += 0.125
    elif case == "long_steps":
        ds, dt = 1.5, 12.0
    elif case == "tiny_negative_offsets":        # fractions 1 - 1e-10, 1 - 3e-10, ...: equal in float arithmetic, not equal
        src = src - rng.choice([1e-10, 3e-10, 7e-10], size=src.shape)
    elif case == "two_warps":
        src = rng.integers(0, 7, (64, 3)).astype(np.float64)
    src = src.astype(np.float32)
    j, k = _random_medium(shape, 1, seed=78)
    ref = oracle_mod.march(j, k, src, n_rays, ds, 1.0, dt, n_steps)
    got = rt.rt_march(_dev(j), _dev(k), _dev(src), n_rays, ds, 1.0, dt, n_steps).cpu().numpy()
    parity.assert_parity(got, ref, f"shared fractions: {case}")
    plain = rt.rt_march_ex(_dev(j), _dev(k), _dev(src), n_rays, ds, 1.0, dt, n_steps, variant=5).cpu().numpy()
    assert np.abs(got - plain).max() <= 1e-6 * np.abs(plain).max()      # same arithmetic per ray, other summation order


@pytest.mark.parametrize("nb,shape", [(3, (9, 7, 8)), (5, (6, 8, 7)), (4, (9, 7, 8)), (8, (7, 9, 6))])
@pytest.mark.parametrize("shared_fractions", [True, False])
def test_bins_with_many_sources(rt, oracle_mod, nb, shape, shared_fractions):
    """>= 32 sources (warp = 32 (source, bin group) pairs x 1 direction) with several bins: bins in fours take the plain
    fp32 scratch with one red.v4 per voxel, other bin counts one bin per lane with fp64 reductions; sources that share
    their cell fractions take the weight-table instantiation, others the plain one.  Three time steps."""
    n_src, n_rays, ds, dt, n_steps = 41, 13, 0.25, 3.0, 3
    rng = np.random.default_rng(nb * 100 + shape[0])
    src = rng.integers(-1, 10, (n_src, 3)).astype(np.float64) + (0.5, 0.25, 0.0)
    if not shared_fractions:
        src += rng.uniform(-0.2, 0.2, src.shape)
    src = src.astype(np.float32)
    j, k = _random_medium(shape, nb, seed=nb)
    ref = oracle_mod.march(j, k, src, n_rays, ds, 1.0, dt, n_steps)
    got = rt.rt_march(_dev(j), _dev(k), _dev(src), n_rays, ds, 1.0, dt, n_steps).cpu().numpy()
    parity.assert_parity(got, ref, f"nb={nb} shared={shared_fractions}")


@pytest.mark.parametrize("shape,nb,n_src,n_rays,dt,n_steps,what", [
    ((48, 40, 44), 4, 5, 301, 4.0, 100, "four bins per thread, sums in the fp32 grid alone (1.1 deposits per element and step)"),
    ((48, 40, 44), 4, 40, 1024, 34.0, 100, "four bins per thread, fp32 scratch drained into the fp64 grid (264 per element)"),
    ((64, 60, 72), 2, 3, 200, 3.0, 61, "two bins: one bin per lane, fp64 reductions"),
    ((64, 60, 72), 2, 1, 1, 3.0, 61, "one ray"),
])
def test_rays_from_the_list_sorted_by_tile(rt, oracle_mod, shape, nb, n_src, n_rays, dt, n_steps, what):
    """Calls whose fp32 snapshots exceed 128 MiB (here through many time steps on a small grid; C4 through its 256^3
    grid) take their rays from the list sorted by tile (rt_ray_sort.cuh), in every deposit mode of that path; the
    launch count says so.  Sources in general position in and around the box, ragged ray counts."""
    assert int(np.prod(shape)) * nb * n_steps * 4 > 128 << 20
    assert rt.rt_launch_count(*shape, n_src, n_rays, nb, n_steps) == (7 if nb % 4 == 0 else 5)
    rng = np.random.default_rng(n_src + n_rays)
    src = rng.uniform(-2.0, max(shape) + 1.0, (n_src, 3)).astype(np.float32)
    j, k = _random_medium(shape, nb, seed=nb + n_src)
    ref = oracle_mod.march(j, k, src, n_rays, 0.5, 1.0, dt, n_steps)
    got = rt.rt_march(_dev(j), _dev(k), _dev(src), n_rays, 0.5, 1.0, dt, n_steps).cpu().numpy()
    parity.assert_parity(got, ref, what)
    kt = rt.rt_march_trilinear_kappa(_dev(j), _dev(k), _dev(src), n_rays, 0.5, 1.0, dt, n_steps).cpu().numpy()
    if n_src * n_rays <= 2000:
        parity.assert_parity(kt, oracle_mod.march(j, k, src, n_rays, 0.5, 1.0, dt, n_steps, kappa_trilinear=True), what + ", trilinear kappa")


def test_more_sources_than_the_sort_handles(rt, oracle_mod):
    """Above 65,536 sources the spatial source sort is skipped (identity order); same field."""
    shape, n_src = (4, 4, 4), 66000
    j, k = _random_medium(shape, 1, seed=3)
    src = np.random.default_rng(4).uniform(-1.0, 4.0, (n_src, 3)).astype(np.float32)
    ref = oracle_mod.march(j, k, src, 1, 0.5, 1.0, 3.0, 1)
    out = rt.rt_march(_dev(j), _dev(k), _dev(src), 1, 0.5, 1.0, 3.0, 1)
    torch.cuda.synchronize()
    parity.assert_parity(out.cpu().numpy(), ref, "66000 sources")


# ------------------------------------------------------------------------------------------------
# trilinear-kappa variant (D18)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("shape,nb,n_src,n_rays,ds,dt", [
    ((5, 4, 3), 3, 2, 7, 0.5, 5.0),
    ((6, 5, 7), 8, 1, 40, 0.5, 8.0),
    ((9, 8, 7), 1, 40, 24, 0.25, 4.0),          # warp = 32 sources x 1 direction
    ((8, 8, 8), 4, 3, 50, 1.7, 13.6),           # steps longer than a cell
])
def test_trilinear_kappa_small_cases(rt, oracle_mod, shape, nb, n_src, n_rays, ds, dt):
    j, k = _random_medium(shape, nb, seed=sum(shape) + nb)
    src = np.random.default_rng(n_src).uniform(-2.0, max(shape) + 1.0, (n_src, 3)).astype(np.float32)
    src[0] = np.round(src[0])
    for n_steps in (1, 3):
        ref = oracle_mod.march(j, k, src, n_rays, ds, 1.0, dt, n_steps, kappa_trilinear=True)
        nn = oracle_mod.march(j, k, src, n_rays, ds, 1.0, dt, n_steps)
        out = rt.rt_march_trilinear_kappa(_dev(j), _dev(k), _dev(src), n_rays, ds, 1.0, dt, n_steps)
        torch.cuda.synchronize()
        parity.assert_parity(out.cpu().numpy(), ref, f"trilinear kappa {shape} nb={nb} steps={n_steps}")
        assert np.abs(nn - ref).max() > 1e-3 * ref.max()        # the two readings really differ here


@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C4"])
def test_trilinear_kappa_configs(rt, oracle_mod, name):
    """C1 in full; stratified source subsets of C2 (40 cell-centred sources x 4,096 rays: warp = 32 sources x 1
    direction in the trilinear-kappa kernel), C3 (40 sources, 8 bins) and C4 (3 sources on the 256^3 x 4 grid, 8 snapshots)."""
    w = config(name)
    count = {"C1": w.n_src, "C2": 40, "C3": 40, "C4": 3}[name]
    src = w.sources if name == "C1" else np.ascontiguousarray(w.sources[_stratified(w.n_src, count)])
    ref = oracle_mod.march(w.j, w.kappa, src, w.n_rays, w.step_size, w.c, w.dt, w.n_steps, kappa_trilinear=True)
    out = rt.rt_march_trilinear_kappa(_dev(w.j), _dev(w.kappa), _dev(src), w.n_rays, w.step_size, w.c, w.dt, w.n_steps)
    torch.cuda.synchronize()
    rows = parity.assert_parity(out.cpu().numpy(), ref, f"trilinear kappa {name}")
    print(rows[-1])


def test_one_source_a_hundred_thousand_rays(rt, oracle_mod):
    """N_Omega far above a warp and not a power of two (ragged last ray band, padded slots), one source."""
    shape, n_rays = (6, 7, 5), 100003
    j, k = _random_medium(shape, 1, seed=9)
    src = np.array([[2.4, 3.1, 1.7]], dtype=np.float32)
    ref = oracle_mod.march(j, k, src, n_rays, 0.5, 1.0, 3.0, 1)
    out = rt.rt_march(_dev(j), _dev(k), _dev(src), n_rays, 0.5, 1.0, 3.0, 1)
    torch.cuda.synchronize()
    parity.assert_parity(out.cpu().numpy(), ref, "100003 rays")


@pytest.mark.parametrize("nb,n_src", [(1, 3), (1, 40), (4, 3), (8, 40)])
@pytest.mark.parametrize("log2_scale", [-100, 90])
def test_emissivities_of_any_magnitude(rt, oracle_mod, nb, n_src, log2_scale):
    """The field is linear in j (eq. (2)) and the weights are formed before they meet j, so j in
    physical units (1e-30 or 1e+27 instead of O(1)) loses nothing: oracle parity at that scale, and the field
    is the O(1) field times the (power of two, hence exact) scale up to the order of the reductions."""
    shape, n_rays = (6, 5, 7), 50
    j, k = _random_medium(shape, nb, seed=11)
    src = np.random.default_rng(12).uniform(-1.0, 7.0, (n_src, 3)).astype(np.float32)
    scale = np.float32(2.0) ** log2_scale
    js = (j * scale).astype(np.float32)
    ref = oracle_mod.march(js, k, src, n_rays, 0.5, 1.0, 5.0, 2)
    got = rt.rt_march(_dev(js), _dev(k), _dev(src), n_rays, 0.5, 1.0, 5.0, 2).cpu().numpy()
    parity.assert_parity(got, ref, f"j x 2^{log2_scale} nb={nb}")
    unit = rt.rt_march(_dev(j), _dev(k), _dev(src), n_rays, 0.5, 1.0, 5.0, 2).cpu().numpy()
    assert np.abs(got / scale - unit).max() <= 1e-6 * np.abs(unit).max()


@pytest.mark.parametrize("nb,n_src", [(1, 2), (1, 33), (4, 2)])
def test_vacuum_and_opaque_cells(rt, oracle_mod, nb, n_src):
    """kappa = 0 (vacuum), kappa ds ~ 1, ~ 20 and ~ 5000 (exp(-kappa ds) underflows to 0 in fp32 and in fp64) mixed
    cell by cell: attenuation factors from 1 down to exactly 0 along one ray."""
    shape, n_rays = (8, 7, 6), 60
    rng = np.random.default_rng(21)
    j = rng.uniform(0.1, 1.0, shape + (nb,)).astype(np.float32)
    k = rng.choice(np.array([0.0, 2.0, 40.0, 1.0e4], dtype=np.float32), size=shape + (nb,), p=[0.4, 0.4, 0.15, 0.05])
    src = rng.uniform(0.0, 6.0, (n_src, 3)).astype(np.float32)
    ref = oracle_mod.march(j, k, src, n_rays, 0.5, 1.0, 6.0, 2)
    got = rt.rt_march(_dev(j), _dev(k), _dev(src), n_rays, 0.5, 1.0, 6.0, 2).cpu().numpy()
    assert np.isfinite(got).all()
    parity.assert_parity(got, ref, f"vacuum/opaque nb={nb} n_src={n_src}")


@pytest.mark.parametrize("nb", [1, 4])
def test_many_time_steps_of_one_substep(rt, oracle_mod, nb):
    """n_steps = 40 snapshots with N_s = 1: every substep is a time-step boundary (flush, next slice)."""
    shape = (6, 6, 6)
    j, k = _random_medium(shape, nb, seed=nb)
    src = np.array([[2.5, 2.5, 2.5], [0.0, 5.0, 3.0]], dtype=np.float32)
    ref = oracle_mod.march(j, k, src, 30, 0.5, 1.0, 0.5, 40)
    out = rt.rt_march(_dev(j), _dev(k), _dev(src), 30, 0.5, 1.0, 0.5, 40)
    torch.cuda.synchronize()
    parity.assert_parity(out.cpu().numpy(), ref, f"40 steps nb={nb}")


def test_out_is_overwritten_and_call_is_repeatable(rt, oracle_mod):
    w = config("C0")
    j, k, s = _dev(w.j), _dev(w.kappa), _dev(w.sources)
    out = torch.full((1,) + w.j.shape, 7.0, device="cuda")
    ws = rt.alloc_workspace(16, 16, 16, 1, w.n_rays, 1, 1)
    for _ in range(3):
        rt.rt_march(j, k, s, w.n_rays, w.step_size, w.c, w.dt, 1, out=out, workspace=ws)
    torch.cuda.synchronize()
    parity.assert_parity(out.cpu().numpy(), oracle_march(oracle_mod, w), "repeat")


@pytest.mark.parametrize("nb,n_src", [(1, 3), (1, 40), (4, 40), (8, 2), (3, 33)])
def test_nothing_is_written_outside_out_workspace_and_state(rt, nb, n_src):
    """Guard bands around every buffer the library writes (compute-sanitizer is closed on this pool): out, the
    workspace and the ray state sit inside larger allocations whose margins must come back untouched."""
    shape, n_rays, ds, dt, n_steps, g = (9, 7, 6), 21, 0.5, 4.0, 3, 4096
    j, k = _random_medium(shape, nb, seed=nb + n_src)
    src = np.random.default_rng(n_src).uniform(-3.0, 12.0, (n_src, 3)).astype(np.float32)
    dj, dk, dsrc = _dev(j), _dev(k), _dev(src)
    n_out = n_steps * j.size
    obuf = torch.full((n_out + 2 * g,), 12345.0, device="cuda")
    wbytes = max(rt.rt_workspace_bytes(*shape, n_src, n_rays, nb, n_steps), rt.rt_step_workspace_bytes(*shape, n_src, n_rays, nb))
    wbuf = torch.full((wbytes + 2 * g,), 0xAB, dtype=torch.uint8, device="cuda")
    sfl = rt.rt_state_bytes(n_src, n_rays, nb) // 4
    sbuf = torch.full((sfl + 2 * g,), 777.0, device="cuda")
    out, ws, state = obuf[g:g + n_out], wbuf[g:g + wbytes], sbuf[g:g + sfl]
    for variant in (0, 1, 4, 5, 16, 32):
        rt.rt_march_ex(dj, dk, dsrc, n_rays, ds, 1.0, dt, n_steps, out=out, workspace=ws, variant=variant)
    rt.rt_state_reset(n_src, n_rays, nb, state=state)
    for m in range(2):
        rt.rt_march_step(dj, dk, dsrc, n_rays, ds, 1.0, dt, m * 8, state, out=out[:j.size], accumulate=bool(m), workspace=ws)
    torch.cuda.synchronize()
    assert (obuf[:g] == 12345.0).all() and (obuf[g + n_out:] == 12345.0).all()
    assert (wbuf[:g] == 0xAB).all() and (wbuf[g + wbytes:] == 0xAB).all()
    assert (sbuf[:g] == 777.0).all() and (sbuf[g + sfl:] == 777.0).all()
    assert torch.isfinite(out).all() and torch.isfinite(state).all()


def test_runs_on_a_side_stream(rt, oracle_mod):
    w = config("C0")
    st = torch.cuda.Stream()
    j, k, s = _dev(w.j), _dev(w.kappa), _dev(w.sources)
    torch.cuda.synchronize()
    with torch.cuda.stream(st):
        out = rt.rt_march(j, k, s, w.n_rays, w.step_size, w.c, w.dt, 1)
    st.synchronize()
    parity.assert_parity(out.cpu().numpy(), oracle_march(oracle_mod, w), "side stream")


def test_error_codes_on_device(rt):
    w = config("C0")
    j, k, s = _dev(w.j), _dev(w.kappa), _dev(w.sources)
    with pytest.raises(rt.RtError) as e:
        rt.rt_march(j, k, s, w.n_rays, w.step_size, w.c, w.dt, 1, workspace=torch.empty(16, dtype=torch.uint8, device="cuda"))
    assert e.value.code == rt.RT_EWORKSPACE
    with pytest.raises(rt.RtError) as e:
        rt.rt_march(j, k, s, 0, w.step_size, w.c, w.dt, 1)
    assert e.value.code == rt.RT_EINVAL
    with pytest.raises(rt.RtError) as e:
        rt.rt_march(j, k, s, w.n_rays, -1.0, w.c, w.dt, 1)
    assert e.value.code == rt.RT_EINVAL


# ------------------------------------------------------------------------------------------------
# C2, C3, C4: oracle parity on stratified source subsets (all other arguments are the config's)
# ------------------------------------------------------------------------------------------------
SUBSETS = {"C2": 48, "C3": 6, "C4": 3}


@pytest.mark.parametrize("name", ["C2", "C3", "C4"])
def test_large_configs_subset_parity(rt, oracle_mod, name):
    w = config(name)
    idx = _stratified(w.n_src, SUBSETS[name])
    src = np.ascontiguousarray(w.sources[idx])
    ref = oracle_march(oracle_mod, w, src)
    for variant in (0, 4, 5):
        got = gpu_march(rt, w, variant, sources=src)
        rows = parity.assert_parity(got, ref, f"{name} subset variant {variant}")
    print(name, "subset parity:", rows[-1])
    # the textbook kernel (8 fp32 reductions per ray-substep straight into the grid) on 3 sources: with more, the
    # clamped boundary voxels receive so many tiny sequential fp32 adds that ITS rounding error, not the
    # method, exceeds the tolerance -- the product kernel pre-sums in registers
    few = src[:3]
    ref_few = oracle_march(oracle_mod, w, few)
    for variant in (1, 2):
        parity.assert_parity(gpu_march(rt, w, variant, sources=few), ref_few, f"{name} 3 sources variant {variant}")


# ------------------------------------------------------------------------------------------------
# full size, the launch configuration bench.py times: properties that hold at any size
# ------------------------------------------------------------------------------------------------
def _close(a, b, what):
    """Two fp32 GPU fields of the same quantity: each is within tolerance of the exact field, so they are
    within twice the tolerance of one another."""
    rows = parity.compare(a, b.astype(np.float64))
    for r in rows:
        assert r["nonfinite"] == 0, (what, r)
        assert r["rel_l2"] <= 2 * parity.REL_L2_TOL and r["max_voxel_rel"] <= 2 * parity.PER_VOXEL_TOL, (what, r)
    return rows


@pytest.mark.parametrize("name", ["C2", "C3", "C4"])
def test_full_size_properties(rt, name):
    w = config(name)
    full = gpu_march(rt, w, 0)
    assert np.isfinite(full).all() and full.min() >= 0.0
    # (1) run-to-run: only the order of the fp32 reductions differs
    _close(gpu_march(rt, w, 0), full, f"{name} rerun")
    # (2) additivity over sources: the sum of chunk fields is the field
    chunks = np.array_split(np.arange(w.n_src), 4)
    parts = sum(gpu_march(rt, w, 0, sources=np.ascontiguousarray(w.sources[c])).astype(np.float64) for c in chunks)
    _close(full, parts, f"{name} additivity")
    # (3) snapshots are cumulative and non-decreasing (D7): deposits are non-negative
    for m in range(1, w.n_steps):
        assert (full[m] >= full[m - 1] * (1 - 1e-6)).all()
    # (4) prefix property (pin P7): the last snapshot's predecessor equals a shorter run's last snapshot
    if w.n_steps > 1:
        short = gpu_march(rt, w, 0, n_steps=w.n_steps - 1)
        _close(short, full[:-1], f"{name} prefix")
    # (5) beyond the light front the field is exactly zero (pin P5): last deposit position + stencil reach
    ax = [np.arange(n, dtype=np.float32) for n in w.shape]
    d2min = np.full(w.shape, np.inf, dtype=np.float32)
    for s in w.sources:
        d2 = ((ax[0] - s[0]) ** 2)[:, None, None] + ((ax[1] - s[1]) ** 2)[None, :, None] + \
             ((ax[2] - s[2]) ** 2)[None, None, :]
        np.minimum(d2min, d2, out=d2min)
    for m in range(w.n_steps):
        reach = ((m + 1) * w.substeps_per_step - 1) * w.step_size + np.sqrt(3.0)
        dark = d2min > np.float32(reach * reach * 1.0001)
        assert np.count_nonzero(full[m][dark]) == 0, (name, m, int(dark.sum()))


def _host_ram_gib():
    try:
        return os.sysconf("SC_PAGE_SIZE") * os.sysconf("SC_PHYS_PAGES") / 2 ** 30
    except (ValueError, OSError):
        return 0.0


@pytest.mark.parametrize("name", ["C2", "C3", "C4"])
def test_full_size_oracle_parity(rt, oracle_mod, name):
    """The launch configuration bench.py times, against the oracle on the WHOLE config (tens of seconds of host
    time per config; C4 needs ~16 GiB of host memory for the per-thread fp64 grids and snapshots)."""
    if os.environ.get("RT_SKIP_FULL_PARITY") == "1":
        pytest.skip("RT_SKIP_FULL_PARITY=1")
    if name == "C4" and _host_ram_gib() < 48:
        pytest.skip("C4 full oracle needs a host with >= 48 GiB")
    w = config(name)
    got = gpu_march(rt, w, 0)
    ref = oracle_march(oracle_mod, w)
    rows = parity.assert_parity(got, ref, f"{name} full")
    print(name, "full parity:", rows)


def test_overlapped_batches_never_lose_a_deposit(rt):
    """The batched multi-bin kernels (RT_VARIANT_SLIDING_BY_SOURCE on C3: what rt_march ran in round 1) march their ray
    batches in pairs, the second grid of a pair launched with programmatic stream serialization over the tail of the
    first, and one drain kernel folds both scratch grids.  The drain must see every deposit of BOTH grids whichever
    finishes first (the second grid waits for the first before it completes): 50 repetitions agree with one another to
    the rounding of the reduction order; a drain that overtook a grid would drop whole batches of deposits."""
    w = config("C3")
    j, k, s = _dev(w.j), _dev(w.kappa), _dev(w.sources)
    ws = rt.alloc_workspace(*w.shape, w.n_src, w.n_rays, w.n_bins, w.n_steps)
    args = (w.n_rays, w.step_size, w.c, w.dt, w.n_steps)
    first = rt.rt_march_ex(j, k, s, *args, workspace=ws, variant=rt.RT_VARIANT_SLIDING_BY_SOURCE).clone()
    scale = float(first.max())
    out = torch.empty_like(first)
    worst = 0.0
    for _ in range(50):
        rt.rt_march_ex(j, k, s, *args, out=out, workspace=ws, variant=rt.RT_VARIANT_SLIDING_BY_SOURCE)
        worst = max(worst, float((out - first).abs().max()) / scale)
    assert worst <= 2e-6, worst


def test_concurrent_drains_never_lose_a_deposit(rt):
    """The product path: every block drains a slice of the fp32 scratch into the fp64 grid (atom.exch) while other
    blocks still reduce into it.  C2 (16 drain rounds over 67,584 blocks) and C3 repeated: the runs agree to the
    rounding of the fp32 sums between two drains (a few 1e-6 at the hottest voxel, a grid corner that takes 1 % of all
    deposits), and the total deposited mass (pin P2) to 1e-6: slices of deposits lost between a read and a zeroing
    would show in both."""
    for name, reps in (("C2", 10), ("C3", 20)):
        w = config(name)
        j, k, s = _dev(w.j), _dev(w.kappa), _dev(w.sources)
        ws = rt.alloc_workspace(*w.shape, w.n_src, w.n_rays, w.n_bins, w.n_steps)
        args = (w.n_rays, w.step_size, w.c, w.dt, w.n_steps)
        first = rt.rt_march(j, k, s, *args, workspace=ws).clone()
        scale = float(first.max())
        total = float(first.double().sum())
        out = torch.empty_like(first)
        for _ in range(reps):
            rt.rt_march(j, k, s, *args, out=out, workspace=ws)
            assert float((out - first).abs().max()) / scale <= 2e-5, name
            assert abs(float(out.double().sum()) - total) <= 1e-6 * total, name
