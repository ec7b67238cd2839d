"""rt_march_step (persistent ray state, the medium may change between time steps; reading D17) against
the fp64 oracle's step entry, element by element, at BASELINE.json's tolerances.  All calls go through the C ABI."""
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


def _media(n, nb, n_steps, seed):
    """A medium per time step: the density field is advected (rolled) and rescaled from step to step."""
    rho = workloads.lognormal_density(n, seed, 1.0)
    ks, js = workloads.bin_scalings(nb)
    out = []
    for m in range(n_steps):
        r = np.roll(rho, shift=(m, 2 * m, -m), axis=(0, 1, 2)) * (1.0 + 0.25 * m)
        out.append((np.ascontiguousarray((1e-3 * r ** 2)[..., None] * js, dtype=np.float32),
                    np.ascontiguousarray((0.05 * r)[..., None] * ks, dtype=np.float32)))
    return out


@pytest.mark.parametrize("n,nb,n_src,n_rays,integer_sources", [
    (20, 1, 3, 64, False),        # few sources: warp = 32 directions of one source
    (20, 1, 40, 48, True),        # warp = 32 sorted sources x 1 direction, cell-centred, ragged last group
    (16, 4, 36, 40, False),       # 4 bins per thread: batched fp32 path with the scratch grid in the workspace
    (16, 8, 2, 33, True),         # 8 bins = 2 bin groups in adjacent lanes
    (12, 3, 5, 20, False),        # bins not a multiple of 4
    (14, 4, 40, 24, True),        # 4 bins per thread, >= 32 cell-centred sources: weight table + plain fp32 scratch
    (12, 3, 33, 20, True),        # 3 bins, one per lane, fp64 reductions, weight table
    (12, 5, 35, 20, False),       # 5 bins, sources in general position
])
def test_steps_with_a_changing_medium_match_the_oracle(rt, oracle_mod, n, nb, n_src, n_rays, integer_sources):
    n_steps, ds, dt = 4, 0.5, 3.0
    media = _media(n, nb, n_steps, seed=100 + n + nb)
    rng = np.random.default_rng(n_src)
    src = rng.uniform(-1.0, n, (n_src, 3))
    src = (np.round(src) if integer_sources else src).astype(np.float32)
    ns = oracle_mod.substeps(ds, 1.0, dt)
    assert rt.rt_substeps_per_step(ds, 1.0, dt) == ns
    ostate = oracle_mod.new_state(n_src, n_rays, nb)
    gstate = rt.rt_state_reset(n_src, n_rays, nb)
    dsrc = _dev(src)
    running = torch.zeros((n, n, n, nb), dtype=torch.float32, device="cuda")
    ref_running = np.zeros((n, n, n, nb))
    for m, (j, k) in enumerate(media):
        ref = oracle_mod.step(j, k, src, n_rays, ds, 1.0, dt, m * ns, ostate)
        before = gstate.clone()
        inc = rt.rt_march_step(_dev(j), _dev(k), dsrc, n_rays, ds, 1.0, dt, m * ns, gstate)
        rt.rt_march_step(_dev(j), _dev(k), dsrc, n_rays, ds, 1.0, dt, m * ns, before, out=running, accumulate=True)
        torch.cuda.synchronize()
        assert torch.equal(before, gstate)             # the carried state does not depend on the accumulate flag
        torch.cuda.synchronize()
        parity.assert_parity(inc.cpu().numpy()[None], ref[None], f"step {m} increment")
        ref_running += ref
        parity.assert_parity(running.cpu().numpy()[None], ref_running[None], f"step {m} accumulated")
        # carried state: I (scaled by 4 pi / N_Omega on the GPU) and exp(-tau)
        g = gstate.cpu().numpy().astype(np.float64)
        scale = 4.0 * np.pi / n_rays
        assert np.abs(g[0] - scale * ostate[:, :, 0, :]).max() <= 2e-5 * scale * ostate[:, :, 0, :].max()
        assert np.abs(g[1] - np.exp(-ostate[:, :, 1, :])).max() <= 2e-5


def test_steps_on_a_c4_shaped_grid_with_a_changing_medium_match_the_oracle(rt, oracle_mod):
    """The branch C4 takes in rt_march_step: a 256^3 x 4-bin grid is too large for the batched fp32 path, so the step
    marches one bin per thread with fp64 reductions into the workspace grid.  C4's own grid, rays, step size and
    substeps per step, 2 of its sources, 3 time steps, the medium advected and rescaled between steps."""
    w = workloads.make_config("C4")
    src = np.ascontiguousarray(w.sources[[5, 41]])
    n, nb, ns = w.shape[0], w.n_bins, w.substeps_per_step
    ostate = oracle_mod.new_state(len(src), w.n_rays, nb)
    gstate = rt.rt_state_reset(len(src), w.n_rays, nb)
    dsrc = _dev(src)
    running = torch.zeros(w.j.shape, dtype=torch.float32, device="cuda")
    ref_running = np.zeros(w.j.shape)
    for m in range(3):
        j = np.ascontiguousarray(np.roll(w.j, shift=(3 * m, -2 * m, m), axis=(0, 1, 2)) * np.float32(1.0 + 0.5 * m))
        k = np.ascontiguousarray(np.roll(w.kappa, shift=(3 * m, -2 * m, m), axis=(0, 1, 2)) * np.float32(1.0 + 0.25 * m))
        ref = oracle_mod.step(j, k, src, w.n_rays, w.step_size, w.c, w.dt, m * ns, ostate)
        rt.rt_march_step(_dev(j), _dev(k), dsrc, w.n_rays, w.step_size, w.c, w.dt, m * ns, gstate, out=running,
                         accumulate=True)
        torch.cuda.synchronize()
        ref_running += ref
        rows = parity.assert_parity(running.cpu().numpy()[None], ref_running[None], f"C4-shaped step {m} accumulated")
        print(rows[-1])
    g = gstate.cpu().numpy().astype(np.float64)
    scale = 4.0 * np.pi / w.n_rays
    assert np.abs(g[0] - scale * ostate[:, :, 0, :]).max() <= 2e-5 * scale * ostate[:, :, 0, :].max()
    assert np.abs(g[1] - np.exp(-ostate[:, :, 1, :])).max() <= 2e-5


def test_steps_in_a_static_medium_reproduce_rt_march(rt, oracle_mod):
    w = workloads.make_config("C1")
    j, k, s = _dev(w.j), _dev(w.kappa), _dev(w.sources)
    snaps = rt.rt_march(j, k, s, w.n_rays, w.step_size, w.c, w.dt, w.n_steps)
    state = rt.rt_state_reset(w.n_src, w.n_rays, 1)
    field = torch.zeros(w.j.shape, dtype=torch.float32, device="cuda")
    for m in range(w.n_steps):
        rt.rt_march_step(j, k, s, w.n_rays, w.step_size, w.c, w.dt, m * w.substeps_per_step, state, out=field,
                         accumulate=True)
        torch.cuda.synchronize()
        a, b = field.cpu().numpy().astype(np.float64), snaps[m].cpu().numpy().astype(np.float64)
        assert np.abs(a - b).max() <= 3e-7 * b.max()       # same per-ray arithmetic; only fp32 rounding of the sums
    ref = oracle_mod.march(w.j, w.kappa, w.sources, w.n_rays, w.step_size, w.c, w.dt, w.n_steps)
    parity.assert_parity(field.cpu().numpy()[None], ref[-1:], "C1 stepped")


def test_step_argument_errors(rt):
    n = 8
    j = torch.zeros((n, n, n, 1), device="cuda")
    s = torch.zeros((1, 3), device="cuda")
    state = rt.rt_state_reset(1, 16, 1)
    with pytest.raises(rt.RtError) as e:
        rt.rt_march_step(j, j, s, 16, 0.5, 1.0, 2.0, -1, state)
    assert e.value.code == rt.RT_EINVAL
    with pytest.raises(rt.RtError) as e:
        rt.rt_march_step(j, j, s, 16, 0.5, 1.0, 2.0, 0, state, workspace=torch.empty(16, dtype=torch.uint8, device="cuda"))
    assert e.value.code == rt.RT_EWORKSPACE
    with pytest.raises(ValueError):
        rt.rt_march_step(j, j, s, 16, 0.5, 1.0, 2.0, 0, torch.zeros(7, device="cuda"))
