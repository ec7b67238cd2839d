"""Thin ctypes binding of ``librtmarch.so`` (``include/rtmarch.h``): argument marshalling only.

Every function has the name of the C entry point it calls.  Device-pointer functions take torch CUDA
tensors (PyTorch is used for device memory and streams, nothing else) and enqueue on torch's current
stream unless ``stream`` is given; ``rt_march_host`` takes numpy arrays.  There is no CPU or PyTorch
fallback: if the library cannot be loaded the import of this module raises.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from . import build as _build

RT_OK, RT_EINVAL, RT_EWORKSPACE, RT_ECUDA, RT_EALIGN = 0, -1, -2, -3, -4
RT_VARIANT_DEFAULT, RT_VARIANT_DIRECT, RT_VARIANT_DIRECT_COHERENT, RT_VARIANT_SLIDING_LATTICE = 0, 1, 2, 3
RT_VARIANT_SLIDING_BY_DIRECTION, RT_VARIANT_SLIDING_BY_SOURCE, RT_VARIANT_FLAG_ACC_F32 = 4, 5, 16
RT_VARIANT_FLAG_ONE_BIN = 32
RED_MODES = {"M1_scalar_random": 0, "M2_v4_random": 1, "M3_stencil": 2, "M4_one_address": 3,
             "M5_coalesced": 4, "M6_stencil_walk": 5, "M1_f64_scalar_random": 6, "M3_f64_stencil": 7,
             "M4_eight_corners": 8, "M4_boundary_shell": 9}

EXPORTS = ("rt_march", "rt_march_single", "rt_march_ex", "rt_march_host", "rt_workspace_bytes",
           "rt_substeps_per_step", "rt_launch_count", "rt_directions", "rt_ray_order", "rt_ray_slots", "rt_trace_ray",
           "rt_bench_red_ceiling", "rt_strerror", "rt_version", "rt_state_bytes", "rt_state_reset",
           "rt_step_workspace_bytes", "rt_march_step", "rt_march_trilinear_kappa", "rt_adjoint_workspace_bytes",
           "rt_march_adjoint_j", "rt_adjoint_kappa_workspace_bytes", "rt_march_adjoint_kappa", "rt_host_release")


class RtError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {rt_strerror(code)} (code {code})")


def _load() -> ctypes.CDLL:
    path = _build.LIB_PATH
    if not os.path.exists(path):
        path = _build.build_library()          # raises if nvcc is missing: no fallback
    elif _build.is_stale():                    # sources newer than the library: rebuild if a compiler is here
        try:
            path = _build.build_library()
        except RuntimeError:
            if os.environ.get("RT_REQUIRE_FRESH_LIB"):
                raise
    L = ctypes.CDLL(path)
    vp, i, f, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_float, ctypes.c_size_t
    march_args = [vp, vp, i, i, i, vp, i, i, i, f, f, f, i, vp]
    L.rt_march.argtypes = march_args + [vp, sz, vp]
    L.rt_march_trilinear_kappa.argtypes = march_args + [vp, sz, vp]
    L.rt_adjoint_workspace_bytes.argtypes = [i] * 7
    L.rt_adjoint_workspace_bytes.restype = sz
    L.rt_march_adjoint_j.argtypes = march_args + [vp, sz, vp]
    L.rt_adjoint_kappa_workspace_bytes.argtypes = [i] * 6 + [f, f, f, i]
    L.rt_adjoint_kappa_workspace_bytes.restype = sz
    L.rt_march_adjoint_kappa.argtypes = [vp] + march_args + [vp, sz, vp]
    L.rt_march_single.argtypes = [vp, vp, i, i, i, vp, i, i, f, f, f, i, vp, vp, sz, vp]
    L.rt_march_ex.argtypes = march_args + [vp, sz, vp, i]
    L.rt_march_host.argtypes = march_args
    L.rt_workspace_bytes.argtypes = [i] * 7
    L.rt_workspace_bytes.restype = sz
    L.rt_substeps_per_step.argtypes = [f, f, f]
    L.rt_launch_count.argtypes = [i] * 7
    L.rt_directions.argtypes = [i, vp, vp]
    L.rt_ray_order.argtypes = [i, vp, vp]
    L.rt_ray_slots.argtypes = [i]
    L.rt_trace_ray.argtypes = [vp, vp, i, i, i, i, vp, i, i, f, i, vp, vp, vp, vp]
    L.rt_bench_red_ceiling.argtypes = [i, vp, i, i, i, i, ctypes.c_longlong, ctypes.c_uint,
                                       ctypes.POINTER(ctypes.c_longlong), vp]
    L.rt_state_bytes.argtypes = [i, i, i]
    L.rt_state_bytes.restype = sz
    L.rt_state_reset.argtypes = [vp, i, i, i, vp]
    L.rt_step_workspace_bytes.argtypes = [i] * 6
    L.rt_step_workspace_bytes.restype = sz
    L.rt_march_step.argtypes = [vp, vp, i, i, i, vp, i, i, i, f, f, f, ctypes.c_longlong, vp, vp, i, vp, sz, vp]
    L.rt_strerror.argtypes = [i]
    L.rt_strerror.restype = ctypes.c_char_p
    L.rt_version.restype = ctypes.c_char_p
    for name in EXPORTS:
        getattr(L, name)                       # AttributeError if the library lacks a declared symbol
    return L


_lib = _load()


def library_path() -> str:
    return _build.LIB_PATH


def rt_strerror(code: int) -> str:
    return _lib.rt_strerror(int(code)).decode()


def rt_version() -> str:
    return _lib.rt_version().decode()


def rt_substeps_per_step(step_size: float, c: float, dt: float) -> int:
    return int(_lib.rt_substeps_per_step(step_size, c, dt))


def rt_workspace_bytes(nx, ny, nz, n_src, n_rays, n_bins, n_steps) -> int:
    return int(_lib.rt_workspace_bytes(nx, ny, nz, n_src, n_rays, n_bins, n_steps))


def rt_launch_count(nx, ny, nz, n_src: int, n_rays: int, n_bins: int, n_steps: int) -> int:
    return int(_lib.rt_launch_count(nx, ny, nz, n_src, n_rays, n_bins, n_steps))


def rt_ray_slots(n_rays: int) -> int:
    return int(_lib.rt_ray_slots(n_rays))


# ---------------------------------------------------------------------------------------------------
# device-pointer entry points (torch tensors carry the memory)
# ---------------------------------------------------------------------------------------------------
def _torch():
    import torch
    return torch


def _stream_ptr(stream):
    if stream is None:
        return _torch().cuda.current_stream().cuda_stream
    return getattr(stream, "cuda_stream", stream)


def _check_dev(t, name, dtype, ndim=None):
    torch = _torch()
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{name}: expected a CUDA torch tensor (there is no CPU path)")
    if t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{name}: expected contiguous {dtype}")
    if ndim is not None and t.dim() != ndim:
        raise ValueError(f"{name}: expected {ndim} dimensions, got {tuple(t.shape)}")
    return t


def alloc_workspace(nx, ny, nz, n_src, n_rays, n_bins, n_steps, device=None):
    torch = _torch()
    n = max(16, rt_workspace_bytes(nx, ny, nz, n_src, n_rays, n_bins, n_steps))
    return torch.empty(n, dtype=torch.uint8, device=device or "cuda")


def rt_march_ex(j, kappa, sources, n_rays, step_size, c, dt, n_steps, out=None, workspace=None, stream=None,
                variant=RT_VARIANT_DEFAULT, _entry=None):
    """out[n_steps,nx,ny,nz,n_bins] = the march of include/rtmarch.h; asynchronous on the stream."""
    torch = _torch()
    _check_dev(j, "j", torch.float32, 4)
    _check_dev(kappa, "kappa", torch.float32, 4)
    _check_dev(sources, "sources", torch.float32, 2)
    if kappa.shape != j.shape or sources.shape[1] != 3:
        raise ValueError("kappa must have j's shape and sources must be [n_src, 3]")
    nx, ny, nz, nb = j.shape
    n_src = sources.shape[0]
    if out is None:
        out = torch.empty((n_steps, nx, ny, nz, nb), dtype=torch.float32, device=j.device)
    else:
        _check_dev(out, "out", torch.float32)
        if out.numel() != n_steps * j.numel():
            raise ValueError("out has the wrong size")
    if workspace is None:
        workspace = alloc_workspace(nx, ny, nz, n_src, n_rays, nb, n_steps, j.device)
    args = (j.data_ptr(), kappa.data_ptr(), nx, ny, nz, sources.data_ptr(), n_src, n_rays, nb, step_size, c, dt,
            n_steps, out.data_ptr(), workspace.data_ptr(), workspace.numel(), _stream_ptr(stream))
    rc = _entry(*args) if _entry is not None else _lib.rt_march_ex(*args, variant)
    if rc != RT_OK:
        raise RtError(rc, "rt_march")
    return out


def rt_march(j, kappa, sources, n_rays, step_size, c, dt, n_steps, out=None, workspace=None, stream=None):
    return rt_march_ex(j, kappa, sources, n_rays, step_size, c, dt, n_steps, out, workspace, stream,
                       RT_VARIANT_DEFAULT)


def rt_march_trilinear_kappa(j, kappa, sources, n_rays, step_size, c, dt, n_steps, out=None, workspace=None,
                             stream=None):
    """rt_march with kappa read trilinearly (D18)."""
    return rt_march_ex(j, kappa, sources, n_rays, step_size, c, dt, n_steps, out, workspace, stream,
                       _entry=_lib.rt_march_trilinear_kappa)


def rt_adjoint_workspace_bytes(nx, ny, nz, n_src, n_rays, n_bins, n_steps) -> int:
    return int(_lib.rt_adjoint_workspace_bytes(nx, ny, nz, n_src, n_rays, n_bins, n_steps))


def rt_march_adjoint_j(gbar, kappa, sources, n_rays, step_size, c, dt, n_steps, grad_j=None, workspace=None,
                       stream=None):
    """grad_j [nx,ny,nz,n_bins] = dL/dj for gbar [n_steps,nx,ny,nz,n_bins] = dL/d out (D19)."""
    torch = _torch()
    _check_dev(gbar, "gbar", torch.float32, 5)
    _check_dev(kappa, "kappa", torch.float32, 4)
    _check_dev(sources, "sources", torch.float32, 2)
    nx, ny, nz, nb = kappa.shape
    if tuple(gbar.shape) != (n_steps, nx, ny, nz, nb) or sources.shape[1] != 3:
        raise ValueError("gbar must be [n_steps, nx, ny, nz, n_bins] and sources [n_src, 3]")
    n_src = sources.shape[0]
    if grad_j is None:
        grad_j = torch.empty((nx, ny, nz, nb), dtype=torch.float32, device=kappa.device)
    else:
        _check_dev(grad_j, "grad_j", torch.float32)
        if grad_j.numel() != kappa.numel():
            raise ValueError("grad_j has the wrong size")
    if workspace is None:
        workspace = torch.empty(max(16, rt_adjoint_workspace_bytes(nx, ny, nz, n_src, n_rays, nb, n_steps)),
                                dtype=torch.uint8, device=kappa.device)
    rc = _lib.rt_march_adjoint_j(gbar.data_ptr(), kappa.data_ptr(), nx, ny, nz, sources.data_ptr(), n_src, n_rays, nb,
                                 step_size, c, dt, n_steps, grad_j.data_ptr(), workspace.data_ptr(), workspace.numel(),
                                 _stream_ptr(stream))
    if rc != RT_OK:
        raise RtError(rc, "rt_march_adjoint_j")
    return grad_j


def rt_adjoint_kappa_workspace_bytes(nx, ny, nz, n_src, n_rays, n_bins, step_size, c, dt, n_steps) -> int:
    return int(_lib.rt_adjoint_kappa_workspace_bytes(nx, ny, nz, n_src, n_rays, n_bins, step_size, c, dt, n_steps))


def rt_march_adjoint_kappa(gbar, j, kappa, sources, n_rays, step_size, c, dt, n_steps, grad_kappa=None, workspace=None,
                           stream=None):
    """grad_kappa [nx,ny,nz,n_bins] = dL/dkappa for gbar [n_steps,nx,ny,nz,n_bins] = dL/d out (D19)."""
    torch = _torch()
    _check_dev(gbar, "gbar", torch.float32, 5)
    _check_dev(j, "j", torch.float32, 4)
    _check_dev(kappa, "kappa", torch.float32, 4)
    _check_dev(sources, "sources", torch.float32, 2)
    nx, ny, nz, nb = kappa.shape
    if tuple(gbar.shape) != (n_steps, nx, ny, nz, nb) or j.shape != kappa.shape or sources.shape[1] != 3:
        raise ValueError("gbar must be [n_steps, nx, ny, nz, n_bins], j like kappa, sources [n_src, 3]")
    n_src = sources.shape[0]
    if grad_kappa is None:
        grad_kappa = torch.empty((nx, ny, nz, nb), dtype=torch.float32, device=kappa.device)
    else:
        _check_dev(grad_kappa, "grad_kappa", torch.float32)
        if grad_kappa.numel() != kappa.numel():
            raise ValueError("grad_kappa has the wrong size")
    if workspace is None:
        workspace = torch.empty(max(16, rt_adjoint_kappa_workspace_bytes(nx, ny, nz, n_src, n_rays, nb, step_size, c, dt,
                                                                         n_steps)),
                                dtype=torch.uint8, device=kappa.device)
    rc = _lib.rt_march_adjoint_kappa(gbar.data_ptr(), j.data_ptr(), kappa.data_ptr(), nx, ny, nz, sources.data_ptr(),
                                     n_src, n_rays, nb, step_size, c, dt, n_steps, grad_kappa.data_ptr(),
                                     workspace.data_ptr(), workspace.numel(), _stream_ptr(stream))
    if rc != RT_OK:
        raise RtError(rc, "rt_march_adjoint_kappa")
    return grad_kappa


def rt_march_single(j, kappa, source_pos, n_rays, step_size, c, dt, n_steps, out=None, workspace=None,
                    stream=None):
    torch = _torch()
    _check_dev(j, "j", torch.float32, 4)
    _check_dev(kappa, "kappa", torch.float32, 4)
    _check_dev(source_pos, "source_pos", torch.float32)
    if source_pos.numel() != 3 or kappa.shape != j.shape:
        raise ValueError("source_pos must hold 3 floats and kappa must have j's shape")
    nx, ny, nz, nb = j.shape
    if out is None:
        out = torch.empty((n_steps, nx, ny, nz, nb), dtype=torch.float32, device=j.device)
    if workspace is None:
        workspace = alloc_workspace(nx, ny, nz, 1, n_rays, nb, n_steps, j.device)
    rc = _lib.rt_march_single(j.data_ptr(), kappa.data_ptr(), nx, ny, nz, source_pos.data_ptr(), n_rays, nb,
                              step_size, c, dt, n_steps, out.data_ptr(), workspace.data_ptr(),
                              workspace.numel(), _stream_ptr(stream))
    if rc != RT_OK:
        raise RtError(rc, "rt_march_single")
    return out


def rt_state_bytes(n_src: int, n_rays: int, n_bins: int) -> int:
    return int(_lib.rt_state_bytes(n_src, n_rays, n_bins))


def rt_step_workspace_bytes(nx, ny, nz, n_src, n_rays, n_bins) -> int:
    return int(_lib.rt_step_workspace_bytes(nx, ny, nz, n_src, n_rays, n_bins))


def rt_state_reset(n_src: int, n_rays: int, n_bins: int, state=None, stream=None):
    """Fresh ray state (I = 0, exp(-tau) = 1): float32 [2, n_src, n_rays, n_bins] on the current device."""
    torch = _torch()
    if state is None:
        state = torch.empty((2, n_src, n_rays, n_bins), dtype=torch.float32, device="cuda")
    _check_dev(state, "state", torch.float32)
    if state.numel() * 4 != rt_state_bytes(n_src, n_rays, n_bins):
        raise ValueError("state has the wrong size")
    rc = _lib.rt_state_reset(state.data_ptr(), n_src, n_rays, n_bins, _stream_ptr(stream))
    if rc != RT_OK:
        raise RtError(rc, "rt_state_reset")
    return state


def rt_march_step(j, kappa, sources, n_rays, step_size, c, dt, k_begin: int, state, out=None, accumulate=False,
                  workspace=None, stream=None):
    """One time step from substep ``k_begin`` in the medium (j, kappa); ``state`` is updated in place.  Returns
    ``out`` [nx,ny,nz,n_bins]: the field deposited during the step (added to ``out`` when ``accumulate``)."""
    torch = _torch()
    _check_dev(j, "j", torch.float32, 4)
    _check_dev(kappa, "kappa", torch.float32, 4)
    _check_dev(sources, "sources", torch.float32, 2)
    _check_dev(state, "state", torch.float32)
    if kappa.shape != j.shape or sources.shape[1] != 3:
        raise ValueError("kappa must have j's shape and sources must be [n_src, 3]")
    nx, ny, nz, nb = j.shape
    n_src = sources.shape[0]
    if state.numel() * 4 != rt_state_bytes(n_src, n_rays, nb):
        raise ValueError("state has the wrong size")
    if out is None:
        if accumulate:
            raise ValueError("accumulate needs the running field in `out`")
        out = torch.empty((nx, ny, nz, nb), dtype=torch.float32, device=j.device)
    else:
        _check_dev(out, "out", torch.float32)
        if out.numel() != j.numel():
            raise ValueError("out has the wrong size")
    if workspace is None:
        workspace = torch.empty(max(16, rt_step_workspace_bytes(nx, ny, nz, n_src, n_rays, nb)), dtype=torch.uint8,
                                device=j.device)
    rc = _lib.rt_march_step(j.data_ptr(), kappa.data_ptr(), nx, ny, nz, sources.data_ptr(), n_src, n_rays, nb,
                            step_size, c, dt, int(k_begin), state.data_ptr(), out.data_ptr(), int(bool(accumulate)),
                            workspace.data_ptr(), workspace.numel(), _stream_ptr(stream))
    if rc != RT_OK:
        raise RtError(rc, "rt_march_step")
    return out


def rt_directions(n_rays: int, stream=None):
    torch = _torch()
    nhat = torch.empty((n_rays, 3), dtype=torch.float64, device="cuda")
    rc = _lib.rt_directions(n_rays, nhat.data_ptr(), _stream_ptr(stream))
    if rc != RT_OK:
        raise RtError(rc, "rt_directions")
    return nhat


def rt_ray_order(n_rays: int, stream=None):
    torch = _torch()
    order = torch.empty(rt_ray_slots(n_rays), dtype=torch.int32, device="cuda")
    rc = _lib.rt_ray_order(n_rays, order.data_ptr(), _stream_ptr(stream))
    if rc != RT_OK:
        raise RtError(rc, "rt_ray_order")
    return order


def rt_trace_ray(j, kappa, source_pos, ray_index: int, n_rays: int, step_size: float, n_sub: int, stream=None):
    """One ray on the GPU, per-substep records: dict(pos=[n_sub,3] f64, I=[n_sub,B] f32, T=[n_sub,B] f32)."""
    torch = _torch()
    _check_dev(j, "j", torch.float32, 4)
    _check_dev(kappa, "kappa", torch.float32, 4)
    _check_dev(source_pos, "source_pos", torch.float32)
    nx, ny, nz, nb = j.shape
    pos = torch.empty((n_sub, 3), dtype=torch.float64, device=j.device)
    tr_i = torch.empty((n_sub, nb), dtype=torch.float32, device=j.device)
    tr_t = torch.empty((n_sub, nb), dtype=torch.float32, device=j.device)
    rc = _lib.rt_trace_ray(j.data_ptr(), kappa.data_ptr(), nx, ny, nz, nb, source_pos.data_ptr(), ray_index, n_rays,
                           step_size, n_sub, pos.data_ptr(), tr_i.data_ptr(), tr_t.data_ptr(), _stream_ptr(stream))
    if rc != RT_OK:
        raise RtError(rc, "rt_trace_ray")
    return {"pos": pos, "I": tr_i, "T": tr_t}


def rt_bench_red_ceiling(mode: int, grid, n_red: int, seed: int = 1, stream=None) -> int:
    """Enqueue one ceiling microbenchmark on ``grid`` [nx,ny,nz,nb] (float32; float64 for modes 6, 7);
    returns the reductions issued."""
    torch = _torch()
    _check_dev(grid, "grid", torch.float64 if mode in (6, 7) else torch.float32, 4)
    nx, ny, nz, nb = grid.shape
    issued = ctypes.c_longlong(0)
    rc = _lib.rt_bench_red_ceiling(mode, grid.data_ptr(), nx, ny, nz, nb, n_red, seed, ctypes.byref(issued),
                                   _stream_ptr(stream))
    if rc != RT_OK:
        raise RtError(rc, "rt_bench_red_ceiling")
    return int(issued.value)


# ---------------------------------------------------------------------------------------------------
# host-pointer entry point (end to end: H2D, march, D2H inside the call)
# ---------------------------------------------------------------------------------------------------
def rt_march_host(j, kappa, sources, n_rays, step_size, c, dt, n_steps, out=None):
    def f32(a, nd):
        a = np.asarray(a)
        if a.dtype != np.float32 or not a.flags.c_contiguous or a.ndim != nd:
            raise TypeError(f"expected a C-contiguous float32 array with {nd} dimensions")
        return a
    j, kappa, sources = f32(j, 4), f32(kappa, 4), f32(sources, 2)
    if kappa.shape != j.shape or sources.shape[1] != 3:
        raise ValueError("kappa must have j's shape and sources must be [n_src, 3]")
    nx, ny, nz, nb = j.shape
    if out is None:
        out = np.empty((n_steps, nx, ny, nz, nb), dtype=np.float32)
    elif out.dtype != np.float32 or not out.flags.c_contiguous or out.size != n_steps * j.size:
        raise TypeError("out: expected C-contiguous float32 of n_steps * j.size elements")
    rc = _lib.rt_march_host(j.ctypes.data, kappa.ctypes.data, nx, ny, nz, sources.ctypes.data, sources.shape[0],
                            n_rays, nb, step_size, c, dt, n_steps, out.ctypes.data)
    if rc != RT_OK:
        raise RtError(rc, "rt_march_host")
    return out


def rt_host_release() -> None:
    """Give back the device memory rt_march_host keeps between calls."""
    _lib.rt_host_release()


def raw():
    """The ctypes library handle (tests exercise error paths with raw pointers through it)."""
    return _lib
