"""rt_march_static (include/rtmarch.h): the march for callers that may not allocate device memory.  Its workspace is a
file-scope __device__ array of RT_STATIC_WORKSPACE_BYTES inside librtmarch.so; every call on a device shares it.

The GPU tests compare its field with rt_march's (caller-owned workspace) on the same inputs, at the tolerances of the
parity tests (tests/parity.py: relative L2 <= 1e-4, per voxel <= 1e-3 above 1e-6 of the maximum) -- the two run the
same kernels, so they differ by the order of the atomic sums only -- on calls in a row with DIFFERENT shapes, so that a
call meets the contents the previous one left in the array.

This file is collected last on purpose (pytest -x: a failure here hides no other test).
"""
import numpy as np
import pytest

import parity
import workloads

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def rt():
    import paper_2511_09389_b200 as rt
    return rt


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def test_static_workspace_limit_is_checked_on_the_host(rt):
    """No GPU needed: a call that does not fit is refused before any CUDA call (fake non-null pointers)."""
    limit = rt.rt_static_workspace_bytes()
    assert limit == 96 << 20
    L = rt.binding.raw()
    p = 0x1000
    assert rt.rt_workspace_bytes(256, 256, 256, 64, 16384, 4, 8) > limit
    assert L.rt_march_static(p, p, 256, 256, 256, p, 64, 16384, 4, 0.5, 1.0, 32.0, 8, p, None) == rt.RT_ETOOBIG
    assert rt.rt_workspace_bytes(128, 128, 128, 256, 4096, 8, 2) > limit
    assert L.rt_march_static(p, p, 128, 128, 128, p, 256, 4096, 8, 0.5, 1.0, 111.0, 2, p, None) == rt.RT_ETOOBIG
    assert L.rt_march_static(None, p, 8, 8, 8, p, 1, 16, 1, 0.5, 1.0, 2.0, 1, p, None) == rt.RT_EINVAL
    assert L.rt_march_static(p, p, 8, 8, 8, p, 1, 16, 1, 0.0, 1.0, 2.0, 1, p, None) == rt.RT_EINVAL
    assert L.rt_march_static(p + 2, p, 8, 8, 8, p, 1, 16, 1, 0.5, 1.0, 2.0, 1, p, None) == rt.RT_EALIGN
    assert "rt_static_workspace_bytes" in rt.rt_strerror(rt.RT_ETOOBIG)
    assert rt.rt_workspace_bytes(128, 128, 128, 2097, 4096, 1, 1) <= limit      # C2 fits


def _cases():
    """(name, j, kappa, sources, n_rays, ds, c, dt, n_steps): three shapes that use the array differently."""
    c1 = workloads.make_config("C1")                       # 64^3, 1 bin, 4 steps: window-brick scratch, weight table
    yield ("C1", c1.j, c1.kappa, c1.sources, c1.n_rays, c1.step_size, c1.c, c1.dt, c1.n_steps)
    rng = np.random.default_rng(20251109)
    shape, nb = (24, 20, 28), 4                            # 4 bins: plain fp32 scratch = out, 41 sources in general position
    j = rng.uniform(0.1, 1.0, shape + (nb,)).astype(np.float32)
    k = rng.uniform(0.0, 0.6, shape + (nb,)).astype(np.float32)
    src = rng.uniform(-2.0, 29.0, (41, 3)).astype(np.float32)
    yield ("24x20x28 x 4 bins", j, k, src, 200, 0.5, 1.0, 6.0, 3)
    c2 = workloads.make_config("C2")                       # the headline's grid and rays, 40 of its sources: 80 MiB of the 96
    pick = np.unique(np.linspace(0, c2.n_src - 1, 40).round().astype(int))
    yield ("C2, 40 sources", c2.j, c2.kappa, np.ascontiguousarray(c2.sources[pick]), c2.n_rays, c2.step_size, c2.c, c2.dt,
           c2.n_steps)


@pytest.mark.gpu
def test_static_workspace_march_matches_rt_march_on_calls_in_a_row(rt):
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device")
    cases = list(_cases())
    dev = [(name, _dev(j), _dev(k), _dev(s), args) for name, j, k, s, *args in cases]
    # the existing path, caller-owned workspace
    want = {name: rt.rt_march(j, k, s, *args).cpu().numpy().astype(np.float64) for name, j, k, s, args in dev}
    torch.cuda.synchronize()
    # the new entry point: every case twice in a row, then the round again -- each call but the first starts on what
    # another call (of the same or of another shape) left in the static array
    order = [0, 0, 1, 1, 2, 2, 0, 1, 2, 0]
    for n, i in enumerate(order):
        name, j, k, s, args = dev[i]
        out = torch.full((args[-1],) + tuple(j.shape), float("nan"), device="cuda")      # the caller's out; overwritten
        got = rt.rt_march_static(j, k, s, *args, out=out)
        assert got.data_ptr() == out.data_ptr()
        torch.cuda.synchronize()
        parity.assert_parity(got.cpu().numpy(), want[name], f"rt_march_static call {n} ({name}) vs rt_march")


@pytest.mark.gpu
def test_static_workspace_march_allocates_no_device_memory(rt):
    """Device memory in use (cudaMemGetInfo, which sees every allocator of the process) does not change across calls
    once the first call has loaded the kernels; and the entry point works on a side stream."""
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device")
    name, j, k, s, *args = next(_cases())
    j, k, s = _dev(j), _dev(k), _dev(s)
    out = torch.empty((args[-1],) + tuple(j.shape), device="cuda")
    ref = rt.rt_march(j, k, s, *args).cpu().numpy().astype(np.float64)
    side = torch.cuda.Stream()
    rt.rt_march_static(j, k, s, *args, out=out)                      # first call: module load, symbol address
    side.wait_stream(torch.cuda.current_stream())                    # (calls that overlap on the GPU would race on the array)
    rt.rt_march_static(j, k, s, *args, out=out, stream=side)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        rt.rt_march_static(j, k, s, *args, out=out, stream=side)
    side.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, (free0, free1)
    parity.assert_parity(out.cpu().numpy(), ref, "rt_march_static on a side stream vs rt_march")
    with pytest.raises(TypeError):
        rt.rt_march_static(j, k, s, *args, out=None)
    big = torch.zeros((96, 96, 96, 8), device="cuda")                # 8 bins x 3 steps at 96^3: beyond the static array
    assert rt.rt_workspace_bytes(96, 96, 96, 1, 64, 8, 3) > rt.rt_static_workspace_bytes()
    with pytest.raises(rt.RtError) as e:
        rt.rt_march_static(big, big, s[:1].contiguous(), 64, 0.5, 1.0, 4.0, 3, out=torch.empty((3, 96, 96, 96, 8), device="cuda"))
    assert e.value.code == rt.RT_ETOOBIG
