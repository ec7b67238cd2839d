"""CPU-side checks of the C-ABI boundary (no compute calls): the library builds for sm_100a, loads, exports
every symbol include/rtmarch.h declares, and rejects bad arguments on the host before touching CUDA."""
import ctypes
import os
import re
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "rtmarch.h")


@pytest.fixture(scope="module")
def rt():
    import paper_2511_09389_b200 as rt
    return rt


def declared_functions():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(rt_[a-z_0-9]+)\s*\(", text)))


def test_header_declares_the_march_entry_points():
    names = declared_functions()
    for must in ("rt_march", "rt_march_single", "rt_march_host", "rt_workspace_bytes", "rt_substeps_per_step",
                 "rt_strerror", "rt_version", "rt_bench_red_ceiling"):
        assert must in names


def test_library_exports_every_declared_symbol(rt):
    lib = ctypes.CDLL(rt.library_path())
    for name in declared_functions():
        assert hasattr(lib, name), f"{name} declared in rtmarch.h but not exported"
    out = subprocess.run(["nm", "-D", "--defined-only", rt.library_path()], capture_output=True, text=True).stdout
    exported = set(re.findall(r"\bT (rt_[a-z_0-9]+)\b", out))
    assert set(declared_functions()) <= exported
    assert sorted(rt.binding.EXPORTS) == declared_functions()


def test_library_holds_sm100a_code_with_vector_reductions(rt):
    sass = subprocess.run(["cuobjdump", "-sass", rt.library_path()], capture_output=True, text=True).stdout
    assert "sm_100a" in sass
    assert "RED.E.ADD.F32.FTZ.RN" in sass or "REDG.E.ADD.F32" in sass
    assert "F32x4" in sass                      # red.global.add.v4.f32 for bin-innermost groups of 4


def test_header_compiles_as_plain_c(tmp_path):
    src = tmp_path / "t.c"
    src.write_text('#include "rtmarch.h"\nint main(void){return RT_OK;}\n')
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-c", str(src),
                    "-o", str(tmp_path / "t.o")], check=True)


def test_host_side_helpers(rt):
    assert rt.rt_version().startswith("rtmarch")
    assert rt.rt_substeps_per_step(0.5, 1.0, 12.0) == 24
    assert rt.rt_substeps_per_step(0.5, 1.0, 222.0) == 444
    assert rt.rt_substeps_per_step(np.float32(0.1), 1.0, np.float32(0.3)) == 3     # fp32 noise in the ratio (D6)
    assert rt.rt_substeps_per_step(0.3, 1.0, 1.0) == 4                             # ceil
    assert rt.rt_substeps_per_step(1.0, 1.0, 1e-3) == 1
    assert rt.rt_substeps_per_step(0.0, 1.0, 1.0) == rt.RT_EINVAL
    assert rt.rt_substeps_per_step(float("nan"), 1.0, 1.0) == rt.RT_EINVAL
    assert rt.rt_substeps_per_step(1e-12, 1.0, 1.0) == rt.RT_EINVAL                # N_s >= 2^31
    assert rt.rt_workspace_bytes(16, 16, 16, 1, 64, 1, 1) >= 64 * 4
    assert rt.rt_workspace_bytes(16, 16, 16, 1, 0, 1, 1) == 0
    assert rt.rt_ray_slots(4096) >= 4096 and rt.rt_ray_slots(0) == rt.RT_EINVAL
    assert rt.rt_launch_count(16, 16, 16, 1, 64, 1, 1) == 3          # ray order, march, snapshots
    assert rt.rt_launch_count(16, 16, 16, 64, 64, 1, 4) == 6         # + source order, fraction test, the other march instantiation
    assert rt.rt_launch_count(128, 128, 128, 256, 4096, 8, 2) == 6
    assert rt.rt_launch_count(256, 256, 256, 64, 16384, 4, 8) == 7          # sorted ray list: key, scan, scatter, state, 2 marches, snapshots
    assert rt.rt_launch_count(256, 256, 256, 64, 16384, 2, 8) == 5          # ... one march
    for code in (0, -1, -2, -3, -4, -99):
        assert isinstance(rt.rt_strerror(code), str) and rt.rt_strerror(code)


def test_argument_errors_are_caught_before_cuda(rt):
    """Fake non-null pointers: an EINVAL/EALIGN/EWORKSPACE return proves no kernel was launched on them."""
    L = rt.binding.raw()
    p = 0x1000
    ok = dict(j=p, kappa=p, nx=8, ny=8, nz=8, sources=p, n_src=1, n_rays=16, n_bins=1, step_size=0.5, c=1.0,
              dt=2.0, n_steps=1, out=p, workspace=p, workspace_bytes=1 << 20, stream=None)

    def call(**kw):
        a = dict(ok, **kw)
        return L.rt_march(a["j"], a["kappa"], a["nx"], a["ny"], a["nz"], a["sources"], a["n_src"], a["n_rays"],
                          a["n_bins"], a["step_size"], a["c"], a["dt"], a["n_steps"], a["out"], a["workspace"],
                          a["workspace_bytes"], a["stream"])

    for bad in (dict(j=None), dict(kappa=None), dict(sources=None), dict(out=None), dict(nx=0), dict(ny=-1),
                dict(nz=0), dict(n_src=0), dict(n_rays=0), dict(n_bins=0), dict(n_steps=0), dict(step_size=0.0),
                dict(step_size=float("inf")), dict(c=-1.0), dict(dt=float("nan")), dict(n_rays=(1 << 30) + 1),
                dict(nx=2048, ny=2048, nz=2048), dict(step_size=1e-9, dt=100.0), dict(n_steps=1 << 30, dt=8.0)):
        assert call(**bad) == rt.RT_EINVAL, bad
    assert call(j=p + 2) == rt.RT_EALIGN
    assert call(workspace=None) == rt.RT_EWORKSPACE
    assert call(workspace_bytes=8) == rt.RT_EWORKSPACE
    assert call(workspace=p + 4) == rt.RT_EWORKSPACE
    assert L.rt_march_host(None, p, 8, 8, 8, p, 1, 16, 1, 0.5, 1.0, 2.0, 1, p) == rt.RT_EINVAL
    assert L.rt_march_ex(p, p, 8, 8, 8, p, 1, 16, 1, 0.5, 1.0, 2.0, 1, p, p, 1 << 20, None, 7) == rt.RT_EINVAL
    assert L.rt_march_ex(p, p, 8, 8, 8, p, 1, 16, 1, 0.5, 1.0, 2.0, 1, p, p, 1 << 20, None, 128) == rt.RT_EINVAL
    assert L.rt_bench_red_ceiling(10, p, 8, 8, 8, 1, 100, 1, None, None) == rt.RT_EINVAL
    assert L.rt_march_step(p, p, 8, 8, 8, p, 1, 16, 1, 0.5, 1.0, 2.0, 0, None, p, 0, p, 1 << 20, None) == rt.RT_EINVAL
    assert L.rt_march_step(p, p, 8, 8, 8, p, 1, 16, 1, 0.5, 1.0, 2.0, 1 << 40, p, p, 0, p, 1 << 20, None) == rt.RT_EINVAL
    assert L.rt_march_step(p, p, 8, 8, 8, p, 1, 16, 1, 0.5, 1.0, 2.0, 0, p, p, 0, p, 64, None) == rt.RT_EWORKSPACE
    assert L.rt_state_reset(None, 1, 1, 1, None) == rt.RT_EINVAL
    assert rt.rt_state_bytes(2, 3, 4) == 2 * 2 * 3 * 4 * 4 and rt.rt_state_bytes(0, 3, 4) == 0
    assert L.rt_directions(0, p, None) == rt.RT_EINVAL
    assert L.rt_ray_order(16, None, None) == rt.RT_EINVAL


def test_binding_refuses_cpu_tensors(rt):
    torch = pytest.importorskip("torch")
    t = torch.zeros((4, 4, 4, 1))
    with pytest.raises(TypeError):
        rt.rt_march(t, t, torch.zeros((1, 3)), 4, 0.5, 1.0, 1.0, 1)


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2511_09389_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", text, flags=re.M), f
                assert "rt_oracle" not in text and "librtoracle" not in text, f
