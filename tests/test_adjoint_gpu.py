"""rt_march_adjoint_j (dL/dj, reading D19) against the fp64 oracle's adjoint, element by
element, and against the forward CUDA march through the transpose identity <A j, g> = <j, A^T g>."""
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


@pytest.mark.parametrize("shape,nb,n_src,n_rays,ds,dt,n_steps", [
    ((4, 4, 4), 1, 1, 1, 0.5, 4.0, 1),            # the axis ray through and out of a 4-cube
    ((5, 4, 3), 3, 2, 7, 0.5, 5.0, 1),            # rays landing exactly on cell planes (rational z_i)
    ((6, 5, 7), 8, 1, 40, 0.5, 8.0, 3),           # source outside the box, three snapshots
    ((9, 8, 7), 1, 40, 24, 0.25, 4.0, 2),         # warp = 32 sources x 1 direction, ragged group
    ((7, 6, 9), 4, 33, 11, 0.5, 4.0, 2),          # 4 bins, cell-centred and duplicate sources
    ((8, 8, 8), 2, 3, 50, 1.7, 13.6, 1),          # steps longer than a cell
])
def test_adjoint_matches_the_oracle(rt, oracle_mod, shape, nb, n_src, n_rays, ds, dt, n_steps):
    rng = np.random.default_rng(sum(shape) + nb + n_src)
    kap = rng.uniform(0.0, 0.6, shape + (nb,)).astype(np.float32)
    src = rng.uniform(-2.0, max(shape) + 1.0, (n_src, 3))
    if n_src > 3:
        src = np.round(src)
        src[1] = src[0]
    src = src.astype(np.float32)
    if n_src == 1 and n_rays == 1:
        src = np.array([[1.0, 2.0, 1.0]], dtype=np.float32)
    gbar = rng.uniform(0.0, 1.0, (n_steps,) + shape + (nb,)).astype(np.float32)      # >= 0: no cancellation in grad
    ref = oracle_mod.adjoint_j(gbar, kap, src, n_rays, ds, 1.0, dt, n_steps)
    got = rt.rt_march_adjoint_j(_dev(gbar), _dev(kap), _dev(src), n_rays, ds, 1.0, dt, n_steps)
    torch.cuda.synchronize()
    parity.assert_parity(got.cpu().numpy()[None], ref[None], f"adjoint {shape} nb={nb} n_src={n_src} steps={n_steps}")


@pytest.mark.parametrize("name,n_sub_src", [("C1", None), ("C2", 96), ("C3", 40)])
def test_adjoint_is_the_transpose_of_the_cuda_march(rt, name, n_sub_src):
    w = workloads.make_config(name)
    src = w.sources if n_sub_src is None else np.ascontiguousarray(
        w.sources[np.unique(np.linspace(0, w.n_src - 1, n_sub_src).round().astype(int))])
    rng = np.random.default_rng(7)
    j = _dev(w.j)
    kap, dsrc = _dev(w.kappa), _dev(src)
    out = rt.rt_march(j, kap, dsrc, w.n_rays, w.step_size, w.c, w.dt, w.n_steps)
    for trial in range(2):
        g = torch.from_numpy(rng.uniform(0.0, 1.0, tuple(out.shape)).astype(np.float32)).cuda()
        grad = rt.rt_march_adjoint_j(g, kap, dsrc, w.n_rays, w.step_size, w.c, w.dt, w.n_steps)
        torch.cuda.synchronize()
        lhs = float((out.double() * g.double()).sum())
        rhs = float((j.double() * grad.double()).sum())
        assert abs(lhs - rhs) <= 2e-5 * abs(lhs), (name, lhs, rhs)


def test_scalar_amplitude_inversion_on_the_gpu(rt):
    """recover A in j = A e0 from a reference field by gradient descent on the MSE, the gradient from
    the adjoint; the minimiser is the closed form <F, I_ref>/<F, F>."""
    w = workloads.make_config("C1")
    e0, kap, src = _dev(w.j), _dev(w.kappa), _dev(w.sources)
    args = (w.n_rays, w.step_size, w.c, w.dt, w.n_steps)
    F = rt.rt_march(e0, kap, src, *args).double()
    noise = torch.from_numpy(np.random.default_rng(1).standard_normal(tuple(F.shape))).cuda()
    I_ref = 1.8 * F + 0.02 * F.max() * noise
    A_star = float((F * I_ref).sum() / (F * F).sum())
    n = F.numel()
    lip = 2.0 * float((F * F).sum()) / n
    A = 0.2
    for _ in range(25):
        resid = (A * F - I_ref)
        grad_j = rt.rt_march_adjoint_j((2.0 * resid / n).float(), kap, src, *args)
        A -= float((e0.double() * grad_j.double()).sum()) / lip
    torch.cuda.synchronize()
    assert abs(A - A_star) <= 2e-4 * abs(A_star), (A, A_star)


def test_adjoint_argument_errors(rt):
    n = 6
    k = torch.zeros((n, n, n, 1), device="cuda")
    g = torch.zeros((1, n, n, n, 1), device="cuda")
    s = torch.zeros((1, 3), device="cuda")
    with pytest.raises(rt.RtError) as e:
        rt.rt_march_adjoint_j(g, k, s, 16, 0.5, 1.0, 2.0, 1, workspace=torch.empty(16, dtype=torch.uint8, device="cuda"))
    assert e.value.code == rt.RT_EWORKSPACE
    with pytest.raises(ValueError):
        rt.rt_march_adjoint_j(g, k, s, 16, 0.5, 1.0, 2.0, 2)


# ------------------------------------------------------------------------------------------------
# dL/dkappa
# ------------------------------------------------------------------------------------------------
def _signed_compare(got, ref, what):
    """Gradients with respect to kappa have both signs and cancel: compare against the largest entry."""
    scale = np.abs(ref).max()
    rel_l2 = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    worst = np.abs(got - ref).max() / scale
    assert np.isfinite(got).all(), what
    assert rel_l2 <= parity.REL_L2_TOL, (what, rel_l2, worst)
    assert worst <= parity.REL_L2_TOL, (what, rel_l2, worst)           # per entry: 1e-4 of the largest entry
    return rel_l2, worst


@pytest.mark.parametrize("shape,nb,n_src,n_rays,ds,dt,n_steps", [
    ((4, 4, 4), 1, 1, 1, 0.5, 4.0, 1),
    ((5, 4, 3), 3, 2, 7, 0.5, 5.0, 1),
    ((6, 5, 7), 8, 1, 40, 0.5, 8.0, 3),
    ((9, 8, 7), 1, 40, 24, 0.25, 4.0, 2),
    ((7, 6, 9), 4, 33, 11, 0.5, 4.0, 2),
    ((8, 8, 8), 2, 3, 50, 1.7, 13.6, 1),
])
def test_kappa_adjoint_matches_the_oracle(rt, oracle_mod, shape, nb, n_src, n_rays, ds, dt, n_steps):
    rng = np.random.default_rng(sum(shape) + nb + n_src)
    kap = rng.uniform(0.0, 0.6, shape + (nb,)).astype(np.float32)
    j = rng.uniform(0.1, 1.0, shape + (nb,)).astype(np.float32)
    src = rng.uniform(-2.0, max(shape) + 1.0, (n_src, 3))
    if n_src > 3:
        src = np.round(src)
        src[1] = src[0]
    src = src.astype(np.float32)
    if n_src == 1 and n_rays == 1:
        src = np.array([[1.0, 2.0, 1.0]], dtype=np.float32)
    gbar = rng.standard_normal((n_steps,) + shape + (nb,)).astype(np.float32)
    ref = oracle_mod.adjoint_kappa(gbar, j, kap, src, n_rays, ds, 1.0, dt, n_steps)
    got = rt.rt_march_adjoint_kappa(_dev(gbar), _dev(j), _dev(kap), _dev(src), n_rays, ds, 1.0, dt, n_steps)
    torch.cuda.synchronize()
    print(_signed_compare(got.cpu().numpy().astype(np.float64), ref, f"kappa adjoint {shape} nb={nb} n_src={n_src}"))


def test_kappa_adjoint_on_c1_against_the_oracle_and_a_directional_difference(rt, oracle_mod):
    w = workloads.make_config("C1")
    rng = np.random.default_rng(5)
    j, kap, src = _dev(w.j), _dev(w.kappa), _dev(w.sources)
    args = (w.n_rays, w.step_size, w.c, w.dt, w.n_steps)
    out = rt.rt_march(j, kap, src, *args)
    g = torch.from_numpy(rng.uniform(0.0, 1.0, tuple(out.shape)).astype(np.float32)).cuda()
    grad = rt.rt_march_adjoint_kappa(g, j, kap, src, *args)
    torch.cuda.synchronize()
    ref = oracle_mod.adjoint_kappa(g.cpu().numpy(), w.j, w.kappa, w.sources, *args)
    print(_signed_compare(grad.cpu().numpy().astype(np.float64), ref, "kappa adjoint C1"))
    # d/d eps L(kappa (1 + eps d)) at 0, by central differences of the CUDA march
    d = torch.from_numpy(rng.uniform(0.5, 1.5, w.kappa.shape).astype(np.float32)).cuda() * kap
    eps = 1e-2

    def loss(k):
        return float((rt.rt_march(j, k.contiguous(), src, *args).double() * g.double()).sum())

    fd = (loss(kap + eps * d) - loss(kap - eps * d)) / (2 * eps)
    an = float((grad.double() * d.double()).sum())
    assert abs(fd - an) <= 2e-3 * abs(an), (fd, an)


# ------------------------------------------------------------------------------------------------
# paths that only exist at size: oracle parity (not GPU-vs-GPU) on stratified subsets of C2 / C3 / C4, and the source-batch
# loop of rt_march_adjoint_kappa (taken when the forward record of all sources exceeds the record limit)
# ------------------------------------------------------------------------------------------------
def _stratified(n_src, count):
    return np.unique(np.linspace(0, n_src - 1, count).round().astype(int))


def test_adjoint_j_at_full_c2_size_is_the_transpose_and_adds_up_over_source_chunks(rt):
    """The launch configuration of the headline (2,097 sources: brick scratch with 16 concurrent drain rounds): the
    transpose identity against the CUDA march, and the gradient of all sources against the sum of the gradients of four
    source chunks (other drain slices, other summation order), voxel by voxel at the parity tolerances."""
    w = workloads.make_config("C2")
    rng = np.random.default_rng(23)
    j, kap, src = _dev(w.j), _dev(w.kappa), _dev(w.sources)
    args = (w.n_rays, w.step_size, w.c, w.dt, w.n_steps)
    out = rt.rt_march(j, kap, src, *args)
    g = torch.from_numpy(rng.uniform(0.0, 1.0, tuple(out.shape)).astype(np.float32)).cuda()
    grad = rt.rt_march_adjoint_j(g, kap, src, *args)
    torch.cuda.synchronize()
    lhs, rhs = float((out.double() * g.double()).sum()), float((j.double() * grad.double()).sum())
    assert abs(lhs - rhs) <= 2e-5 * abs(lhs), (lhs, rhs)
    parts = torch.zeros_like(grad, dtype=torch.float64)
    for chunk in np.array_split(np.arange(w.n_src), 4):
        parts += rt.rt_march_adjoint_j(g, kap, _dev(w.sources[chunk]), *args).double()
    parity.assert_parity(grad.cpu().numpy()[None], parts.cpu().numpy()[None], "adjoint_j full C2 vs 4 source chunks")


@pytest.mark.parametrize("name,count", [("C2", 40), ("C3", 36), ("C4", 2)])
def test_adjoint_j_on_config_subsets_matches_the_oracle(rt, oracle_mod, name, count):
    """rt_march_adjoint_j with the config's own grid, rays, substeps, steps and bins on a stratified subset of its
    sources (the adjoint is a plain sum over sources, like the field): >= 32 cell-centred sources for C2 / C3 (warp =
    32 sources x 1 direction), 2 of C4's random sources on the 256^3 x 4 grid with 8 snapshots (suffix sums)."""
    w = workloads.make_config(name)
    src = np.ascontiguousarray(w.sources[_stratified(w.n_src, count)])
    rng = np.random.default_rng(11)
    gbar = rng.uniform(0.0, 1.0, (w.n_steps,) + w.j.shape).astype(np.float32)
    got = rt.rt_march_adjoint_j(_dev(gbar), _dev(w.kappa), _dev(src), w.n_rays, w.step_size, w.c, w.dt, w.n_steps)
    torch.cuda.synchronize()
    got = got.cpu().numpy()
    ref = oracle_mod.adjoint_j(gbar, w.kappa, src, w.n_rays, w.step_size, w.c, w.dt, w.n_steps)
    rows = parity.assert_parity(got[None], ref[None], f"adjoint_j {name} subset of {len(src)} sources")
    print(name, rows[-1])


@pytest.mark.parametrize("n_src,n_rays,nb,limit_sources", [
    (70, 24, 1, 32),        # warp = 32 sources x 1 direction: batches of 32, 32 and a ragged 6
    (100, 11, 2, 64),       # two bins: batches of 64 and 36
    (5, 40, 1, 2),          # fewer than 32 sources (warp = 32 directions of one source): batches of 2, 2, 1
])
def test_kappa_adjoint_source_batches_match_the_oracle(rt, oracle_mod, n_src, n_rays, nb, limit_sources):
    """The source-batch loop of rt_march_adjoint_kappa (src_begin offsets, the record stride of each batch, reuse of
    the record buffer), forced on a small case by a record limit of `limit_sources` sources' worth of record
    (rt_march_adjoint_kappa_ex): against the oracle entry by entry, and against the one-batch call."""
    shape, ds, dt, n_steps = (9, 8, 7), 0.25, 4.0, 2
    rng = np.random.default_rng(n_src + nb)
    kap = rng.uniform(0.0, 0.6, shape + (nb,)).astype(np.float32)
    j = rng.uniform(0.1, 1.0, shape + (nb,)).astype(np.float32)
    src = rng.uniform(-2.0, 10.0, (n_src, 3))
    src[: n_src // 2] = np.round(src[: n_src // 2])
    src = src.astype(np.float32)
    gbar = rng.standard_normal((n_steps,) + shape + (nb,)).astype(np.float32)
    K = rt.rt_substeps_per_step(ds, 1.0, dt) * n_steps
    slots = rt.rt_ray_slots(n_rays)
    if n_src >= 32:     # record bytes of one batch = blocks(4 direction slots x 32 (source, bin) pairs) x 128 threads x K x 4
        blocks = ((slots + 3) // 4) * ((limit_sources * nb + 31) // 32)
    else:
        blocks = ((slots * nb + 127) // 128) * limit_sources
    limit = blocks * 128 * K * 4
    args = (_dev(gbar), _dev(j), _dev(kap), _dev(src), n_rays, ds, 1.0, dt, n_steps)
    one = rt.rt_march_adjoint_kappa(*args)
    ws_one = rt.rt_adjoint_kappa_workspace_bytes(*shape, n_src, n_rays, nb, ds, 1.0, dt, n_steps)
    ws_many = rt.rt_adjoint_kappa_workspace_bytes_ex(*shape, n_src, n_rays, nb, ds, 1.0, dt, n_steps, limit)
    assert ws_many < ws_one                                   # the record buffer holds one batch only
    many = rt.rt_march_adjoint_kappa_ex(*args, record_limit=limit)
    torch.cuda.synchronize()
    ref = oracle_mod.adjoint_kappa(gbar, j, kap, src, n_rays, ds, 1.0, dt, n_steps)
    print(_signed_compare(many.cpu().numpy().astype(np.float64), ref, f"kappa adjoint, batches of {limit_sources} of {n_src}"))
    print(_signed_compare(one.cpu().numpy().astype(np.float64), ref, f"kappa adjoint, one batch of {n_src}"))
    scale = float(one.abs().max())
    assert float((one - many).abs().max()) <= 2e-6 * scale    # same per-ray arithmetic, other order of the fp64 sums


def test_kappa_adjoint_c2_subset_in_batches_matches_the_oracle(rt, oracle_mod):
    """C2's grid, rays and substeps with 72 of its sources: the record of all of them (72 x 4,096 x 444 x 8 B = 1 GB)
    is cut into batches of 32 sources by the record limit, as the full config is cut by the 8 GiB default."""
    w = workloads.make_config("C2")
    src = np.ascontiguousarray(w.sources[_stratified(w.n_src, 72)])
    rng = np.random.default_rng(13)
    gbar = rng.uniform(0.0, 1.0, (w.n_steps,) + w.j.shape).astype(np.float32)
    K = w.n_steps * w.substeps_per_step
    limit = (rt.rt_ray_slots(w.n_rays) // 4) * 128 * K * 4               # one group of 32 sources
    got = rt.rt_march_adjoint_kappa_ex(_dev(gbar), _dev(w.j), _dev(w.kappa), _dev(src), w.n_rays, w.step_size, w.c, w.dt,
                                       w.n_steps, record_limit=limit)
    torch.cuda.synchronize()
    ref = oracle_mod.adjoint_kappa(gbar, w.j, w.kappa, src, w.n_rays, w.step_size, w.c, w.dt, w.n_steps)
    print(_signed_compare(got.cpu().numpy().astype(np.float64), ref, "kappa adjoint C2, 72 sources in 3 batches"))


def test_relative_mse_amplitude_inversion_on_the_gpu(rt):
    """PAPER.md:62 names two losses.  The relative MSE weights every voxel by 1 / (I_ref^2 + eps^2) (D20): still
    a parabola in A, minimiser <w F, I_ref> / <w F, F>; the gradient comes from the same adjoint with gbar = 2 w r / n."""
    w = workloads.make_config("C1")
    e0, kap, src = _dev(w.j), _dev(w.kappa), _dev(w.sources)
    args = (w.n_rays, w.step_size, w.c, w.dt, w.n_steps)
    F = rt.rt_march(e0, kap, src, *args).double()
    noise = torch.from_numpy(np.random.default_rng(2).standard_normal(tuple(F.shape))).cuda()
    I_ref = 1.8 * F * (1.0 + 0.05 * noise)
    eps = 1e-3 * float(I_ref.max())
    wgt = 1.0 / (I_ref * I_ref + eps * eps)
    A_star = float((wgt * F * I_ref).sum() / (wgt * F * F).sum())
    n = F.numel()
    lip = 2.0 * float((wgt * F * F).sum()) / n
    A = 0.2
    for _ in range(25):
        resid = A * F - I_ref
        grad_j = rt.rt_march_adjoint_j((2.0 * wgt * resid / n).float(), kap, src, *args)
        A -= float((e0.double() * grad_j.double()).sum()) / lip
    torch.cuda.synchronize()
    assert abs(A - A_star) <= 2e-4 * abs(A_star), (A, A_star)
    plain = float((F * I_ref).sum() / (F * F).sum())
    assert abs(plain - A_star) > 1e-4 * abs(A_star)        # the weighting matters: another minimiser than the plain MSE's


# ------------------------------------------------------------------------------------------------
# forward mode: rt_march_jvp_kappa (D21)
# ------------------------------------------------------------------------------------------------
def _tangent_compare(got, ref, what):
    """A tangent field has both signs (more absorption: less field; a negative dkappa: more): every snapshot against
    the largest entry of the oracle's, like the kappa gradient."""
    for m in range(ref.shape[0]):
        scale = np.abs(ref[m]).max()
        rel_l2 = np.linalg.norm(got[m] - ref[m]) / np.linalg.norm(ref[m])
        worst = np.abs(got[m] - ref[m]).max() / scale
        assert np.isfinite(got[m]).all(), what
        assert rel_l2 <= parity.REL_L2_TOL and worst <= parity.REL_L2_TOL, (what, m, rel_l2, worst)
    return rel_l2, worst


@pytest.mark.parametrize("shape,nb,n_src,n_rays,ds,dt,n_steps,integer_sources", [
    ((4, 4, 4), 1, 1, 1, 0.5, 4.0, 1, True),           # the axis ray through and out of a 4-cube
    ((5, 4, 3), 3, 2, 7, 0.5, 5.0, 1, False),          # 3 bins: one bin per lane, fp64 reductions
    ((6, 5, 7), 8, 1, 40, 0.5, 8.0, 3, False),         # source outside the box, three snapshots
    ((9, 8, 7), 1, 40, 24, 0.25, 4.0, 2, True),        # warp = 32 sources x 1 direction, weight table, brick scratch
    ((9, 8, 7), 1, 45, 24, 0.25, 4.0, 2, False),       # the same in general position (plain instantiation)
    ((7, 6, 9), 4, 33, 11, 0.5, 4.0, 2, True),         # 4 bins
    ((64, 60, 72), 2, 3, 200, 0.5, 3.0, 61, False),    # 135 MB of fp32 snapshots: rays from the list sorted by tile
])
def test_jvp_kappa_matches_the_oracle(rt, oracle_mod, shape, nb, n_src, n_rays, ds, dt, n_steps, integer_sources):
    rng = np.random.default_rng(sum(shape) + nb + n_src)
    kap = rng.uniform(0.0, 0.6, shape + (nb,)).astype(np.float32)
    j = rng.uniform(0.1, 1.0, shape + (nb,)).astype(np.float32)
    dk = rng.uniform(-1.0, 1.0, shape + (nb,)).astype(np.float32)
    src = rng.uniform(-2.0, max(shape) + 1.0, (n_src, 3))
    if integer_sources:
        src = np.round(src)
    src = src.astype(np.float32)
    if n_src == 1 and n_rays == 1:
        src = np.array([[1.0, 2.0, 1.0]], dtype=np.float32)
    ref = oracle_mod.jvp_kappa(j, kap, dk, src, n_rays, ds, 1.0, dt, n_steps)
    got = rt.rt_march_jvp_kappa(_dev(j), _dev(kap), _dev(dk), _dev(src), n_rays, ds, 1.0, dt, n_steps)
    torch.cuda.synchronize()
    print(_tangent_compare(got.cpu().numpy().astype(np.float64), ref, f"jvp {shape} nb={nb} n_src={n_src}"))


def test_jvp_kappa_on_c1_is_dual_to_the_kappa_adjoint_and_matches_a_difference_quotient(rt, oracle_mod):
    """C1 in full against the oracle; <g, J dkappa> = <J^T g, dkappa> with J^T g from rt_march_adjoint_kappa; and the
    paper's global kappa scale (dkappa = kappa) against a central difference of the CUDA march."""
    w = workloads.make_config("C1")
    rng = np.random.default_rng(17)
    j, kap, src = _dev(w.j), _dev(w.kappa), _dev(w.sources)
    args = (w.n_rays, w.step_size, w.c, w.dt, w.n_steps)
    dk = (w.kappa * rng.uniform(0.5, 1.5, w.kappa.shape)).astype(np.float32)
    tang = rt.rt_march_jvp_kappa(j, kap, _dev(dk), src, *args)
    torch.cuda.synchronize()
    ref = oracle_mod.jvp_kappa(w.j, w.kappa, dk, w.sources, *args)
    print(_tangent_compare(tang.cpu().numpy().astype(np.float64), ref, "jvp C1"))
    g = torch.from_numpy(rng.uniform(0.0, 1.0, tuple(tang.shape)).astype(np.float32)).cuda()
    grad = rt.rt_march_adjoint_kappa(g, j, kap, src, *args)
    lhs = float((g.double() * tang.double()).sum())
    rhs = float((grad.double() * _dev(dk).double()).sum())
    assert abs(lhs - rhs) <= 2e-5 * abs(lhs), (lhs, rhs)
    scale = rt.rt_march_jvp_kappa(j, kap, kap, src, *args).double()            # d/d theta of rt_march(j, theta kappa) at 1
    eps = 1e-2
    fd = (rt.rt_march(j, (kap * (1 + eps)).contiguous(), src, *args).double() -
          rt.rt_march(j, (kap * (1 - eps)).contiguous(), src, *args).double()) / (2 * eps)
    assert float((scale - fd).abs().max()) <= 2e-3 * float(fd.abs().max())


def test_kappa_adjoint_and_tangent_are_dual_at_full_c2_size(rt):
    """The launch configurations bench.py times: all 2,097 sources of C2 -- the kappa adjoint in the two source batches
    its 8 GiB record limit gives (15 GB of 4-byte records), the tangent with 16 drain rounds.  <g, J dkappa> =
    <J^T g, dkappa> for a random g and a random positive dkappa ties the two together at that size."""
    w = workloads.make_config("C2")
    rng = np.random.default_rng(29)
    j, kap, src = _dev(w.j), _dev(w.kappa), _dev(w.sources)
    args = (w.n_rays, w.step_size, w.c, w.dt, w.n_steps)
    dk = _dev((w.kappa * rng.uniform(0.5, 1.5, w.kappa.shape)).astype(np.float32))
    tang = rt.rt_march_jvp_kappa(j, kap, dk, src, *args)
    g = torch.from_numpy(rng.uniform(0.0, 1.0, tuple(tang.shape)).astype(np.float32)).cuda()
    grad = rt.rt_march_adjoint_kappa(g, j, kap, src, *args)
    torch.cuda.synchronize()
    assert torch.isfinite(grad).all() and torch.isfinite(tang).all()
    lhs = float((g.double() * tang.double()).sum())
    rhs = float((grad.double() * dk.double()).sum())
    assert abs(lhs - rhs) <= 5e-6 * abs(lhs), (lhs, rhs)          # measured: 5.5e-7


def test_jvp_kappa_on_a_c2_subset(rt, oracle_mod):
    """C2's grid, rays and substeps, 40 of its cell-centred sources: the launch shape of the headline (weight table,
    brick scratch, drains) carrying the tangent."""
    w = workloads.make_config("C2")
    src = np.ascontiguousarray(w.sources[_stratified(w.n_src, 40)])
    got = rt.rt_march_jvp_kappa(_dev(w.j), _dev(w.kappa), _dev(w.kappa), _dev(src), w.n_rays, w.step_size, w.c, w.dt, w.n_steps)
    torch.cuda.synchronize()
    ref = oracle_mod.jvp_kappa(w.j, w.kappa, w.kappa, src, w.n_rays, w.step_size, w.c, w.dt, w.n_steps)
    print(_tangent_compare(got.cpu().numpy().astype(np.float64), ref, "jvp C2 subset"))


def test_jvp_argument_errors(rt):
    n = 6
    k = torch.zeros((n, n, n, 1), device="cuda")
    s = torch.zeros((1, 3), device="cuda")
    with pytest.raises(rt.RtError) as e:
        rt.rt_march_jvp_kappa(k, k, k, s, 16, 1.5, 1.0, 3.0, 1)              # substeps of a cell or more: not offered
    assert e.value.code == rt.RT_EINVAL
    with pytest.raises(ValueError):
        rt.rt_march_jvp_kappa(k, k, torch.zeros((n, n, n, 2), device="cuda"), s, 16, 0.5, 1.0, 2.0, 1)
