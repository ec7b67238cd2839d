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

RT_OK, RT_EINVAL, RT_EWORKSPACE, RT_ECUDA, RT_EALIGN, RT_ETOOBIG = 0, -1, -2, -3, -4, -5
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
           "rt_march_adjoint_j", "rt_adjoint_kappa_workspace_bytes", "rt_march_adjoint_kappa",
           "rt_adjoint_kappa_workspace_bytes_ex", "rt_march_adjoint_kappa_ex", "rt_march_jvp_kappa", "rt_host_release",
           "rt_march_static", "rt_static_workspace_bytes")


class RtError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {rt_strerror(code)} (code {code})")


def _load() -> ctypes.CDLL:
    path = _build.LIB_PATH
    if not os.path.exists(path):
        path = _build.build_library()          # raises if nvcc is missing: no fallback
    elif _build.is_stale():                    # sources newer than the library: rebuild, or fail -- never run stale
        try:                                   # code silently (RT_ALLOW_STALE_LIB=1 overrides, for a box without nvcc)
            path = _build.build_library()
        except RuntimeError:
            if not os.environ.get("RT_ALLOW_STALE_LIB"):
                raise
    L = ctypes.CDLL(path)
    vp, i, f, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_float, ctypes.c_size_t
    march_args = [vp, vp, i, i, i, vp, i, i, i, f, f, f, i, vp]
    L.rt_march.argtypes = march_args + [vp, sz, vp]
    L.rt_march_trilinear_kappa.argtypes = march_args + [vp, sz, vp]
    L.rt_march_static.argtypes = march_args + [vp]
    L.rt_static_workspace_bytes.argtypes = []
    L.rt_static_workspace_bytes.restype = sz
    L.rt_adjoint_workspace_bytes.argtypes = [i] * 7
    L.rt_adjoint_workspace_bytes.restype = sz
    L.rt_march_adjoint_j.argtypes = march_args + [vp, sz, vp]
    L.rt_adjoint_kappa_workspace_bytes.argtypes = [i] * 6 + [f, f, f, i]
    L.rt_adjoint_kappa_workspace_bytes.restype = sz
    L.rt_march_adjoint_kappa.argtypes = [vp] + march_args + [vp, sz, vp]
    L.rt_adjoint_kappa_workspace_bytes_ex.argtypes = [i] * 6 + [f, f, f, i, sz]
    L.rt_adjoint_kappa_workspace_bytes_ex.restype = sz
    L.rt_march_adjoint_kappa_ex.argtypes = [vp] + march_args + [vp, sz, vp, sz]
    L.rt_march_jvp_kappa.argtypes = [vp, vp, vp, i, i, i, vp, i, i, i, f, f, f, i, vp, vp, sz, vp]
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


def _stream_ptr(stream, device=None):
    """cudaStream_t of ``stream`` (a torch stream or a raw handle), else torch's current stream ON ``device``."""
    if stream is None:
        return _torch().cuda.current_stream(device).cuda_stream
    return getattr(stream, "cuda_stream", stream)


class _Call:
    """Context of one device call: makes the tensors' device current (the library launches on the current CUDA
    device) and resolves the stream there.  ``scratch()`` allocates a buffer the call owns: if the launch stream is
    not torch's current stream the buffer is recorded on it, so the caching allocator cannot hand the block to
    another allocation while the enqueued kernels still use it."""

    def __init__(self, stream, *tensors):
        torch = _torch()
        self.device = tensors[0].device
        for t in tensors:
            if t is not None and t.device != self.device:
                raise ValueError(f"all tensors must be on one CUDA device: {t.device} vs {self.device}")
        self._guard = torch.cuda.device(self.device)
        self._stream = stream

    def __enter__(self):
        self._guard.__enter__()
        self.stream_ptr = _stream_ptr(self._stream, self.device)
        return self

    def __exit__(self, *exc):
        return self._guard.__exit__(*exc)

    def scratch(self, shape, dtype):
        torch = _torch()
        t = torch.empty(shape, dtype=dtype, device=self.device)
        cur = torch.cuda.current_stream(self.device)
        if self.stream_ptr != cur.cuda_stream:
            t.record_stream(torch.cuda.ExternalStream(self.stream_ptr, device=self.device))
        return t


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


def _out_or_new(call, out, shape, name):
    """The caller's ``out`` (validated: float32, contiguous, on the call's device, right size) or a fresh one."""
    torch = _torch()
    n = 1
    for d in shape:
        n *= d
    if out is None:
        return call.scratch(shape, torch.float32)
    _check_dev(out, name, torch.float32)
    if out.device != call.device:
        raise ValueError(f"{name} is on {out.device}, the inputs on {call.device}")
    if out.numel() != n:
        raise ValueError(f"{name} has the wrong size")
    return out


def _workspace_or_new(call, workspace, nbytes):
    torch = _torch()
    if workspace is None:
        return call.scratch((max(16, nbytes),), torch.uint8)
    _check_dev(workspace, "workspace", torch.uint8)
    if workspace.device != call.device:
        raise ValueError(f"workspace is on {workspace.device}, the inputs on {call.device}")
    return workspace


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
    with _Call(stream, j, kappa, sources) as call:
        out = _out_or_new(call, out, (n_steps, nx, ny, nz, nb), "out")
        workspace = _workspace_or_new(call, workspace, rt_workspace_bytes(nx, ny, nz, n_src, n_rays, nb, n_steps))
        args = (j.data_ptr(), kappa.data_ptr(), nx, ny, nz, sources.data_ptr(), n_src, n_rays, nb, step_size, c, dt,
                n_steps, out.data_ptr(), workspace.data_ptr(), workspace.numel(), call.stream_ptr)
        rc = _entry(*args) if _entry is not None else _lib.rt_march_ex(*args, variant)
    if rc != RT_OK:
        raise RtError(rc, "rt_march")
    return out


def rt_march(j, kappa, sources, n_rays, step_size, c, dt, n_steps, out=None, workspace=None, stream=None):
    return rt_march_ex(j, kappa, sources, n_rays, step_size, c, dt, n_steps, out, workspace, stream,
                       RT_VARIANT_DEFAULT)


def rt_static_workspace_bytes() -> int:
    return int(_lib.rt_static_workspace_bytes())


def rt_march_static(j, kappa, sources, n_rays, step_size, c, dt, n_steps, out, stream=None):
    """rt_march with the library's static device workspace (include/rtmarch.h): nothing is allocated, here or in the
    library, so ``out`` is the caller's.  Calls that overlap on the GPU race on that workspace."""
    torch = _torch()
    _check_dev(j, "j", torch.float32, 4)
    _check_dev(kappa, "kappa", torch.float32, 4)
    _check_dev(sources, "sources", torch.float32, 2)
    if kappa.shape != j.shape or sources.shape[1] != 3:
        raise ValueError("kappa must have j's shape and sources must be [n_src, 3]")
    if out is None:
        raise TypeError("rt_march_static allocates nothing: pass out")
    nx, ny, nz, nb = j.shape
    with _Call(stream, j, kappa, sources) as call:
        out = _out_or_new(call, out, (n_steps, nx, ny, nz, nb), "out")
        rc = _lib.rt_march_static(j.data_ptr(), kappa.data_ptr(), nx, ny, nz, sources.data_ptr(), sources.shape[0], n_rays, nb,
                                  step_size, c, dt, n_steps, out.data_ptr(), call.stream_ptr)
    if rc != RT_OK:
        raise RtError(rc, "rt_march_static")
    return out


def rt_march_trilinear_kappa(j, kappa, sources, n_rays, step_size, c, dt, n_steps, out=None, workspace=None,
                             stream=None):
    """rt_march with kappa read trilinearly (D18)."""
    return rt_march_ex(j, kappa, sources, n_rays, step_size, c, dt, n_steps, out, workspace, stream,
                       _entry=_lib.rt_march_trilinear_kappa)


def rt_march_jvp_kappa(j, kappa, dkappa, sources, n_rays, step_size, c, dt, n_steps, tangent=None, workspace=None,
                       stream=None):
    """tangent[n_steps,nx,ny,nz,n_bins] = d/d eps rt_march(j, kappa + eps dkappa) at eps = 0 (D21)."""
    torch = _torch()
    _check_dev(j, "j", torch.float32, 4)
    _check_dev(kappa, "kappa", torch.float32, 4)
    _check_dev(dkappa, "dkappa", torch.float32, 4)
    _check_dev(sources, "sources", torch.float32, 2)
    if kappa.shape != j.shape or dkappa.shape != j.shape or sources.shape[1] != 3:
        raise ValueError("kappa and dkappa must have j's shape and sources must be [n_src, 3]")
    nx, ny, nz, nb = j.shape
    n_src = sources.shape[0]
    with _Call(stream, j, kappa, dkappa, sources) as call:
        tangent = _out_or_new(call, tangent, (n_steps, nx, ny, nz, nb), "tangent")
        workspace = _workspace_or_new(call, workspace, rt_workspace_bytes(nx, ny, nz, n_src, n_rays, nb, n_steps))
        rc = _lib.rt_march_jvp_kappa(j.data_ptr(), kappa.data_ptr(), dkappa.data_ptr(), nx, ny, nz, sources.data_ptr(), n_src,
                                     n_rays, nb, step_size, c, dt, n_steps, tangent.data_ptr(), workspace.data_ptr(),
                                     workspace.numel(), call.stream_ptr)
    if rc != RT_OK:
        raise RtError(rc, "rt_march_jvp_kappa")
    return tangent


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
    with _Call(stream, gbar, kappa, sources) as call:
        grad_j = _out_or_new(call, grad_j, (nx, ny, nz, nb), "grad_j")
        workspace = _workspace_or_new(call, workspace, rt_adjoint_workspace_bytes(nx, ny, nz, n_src, n_rays, nb, n_steps))
        rc = _lib.rt_march_adjoint_j(gbar.data_ptr(), kappa.data_ptr(), nx, ny, nz, sources.data_ptr(), n_src, n_rays,
                                     nb, step_size, c, dt, n_steps, grad_j.data_ptr(), workspace.data_ptr(),
                                     workspace.numel(), call.stream_ptr)
    if rc != RT_OK:
        raise RtError(rc, "rt_march_adjoint_j")
    return grad_j


def rt_adjoint_kappa_workspace_bytes(nx, ny, nz, n_src, n_rays, n_bins, step_size, c, dt, n_steps) -> int:
    return int(_lib.rt_adjoint_kappa_workspace_bytes(nx, ny, nz, n_src, n_rays, n_bins, step_size, c, dt, n_steps))


def rt_adjoint_kappa_workspace_bytes_ex(nx, ny, nz, n_src, n_rays, n_bins, step_size, c, dt, n_steps,
                                        record_limit: int) -> int:
    return int(_lib.rt_adjoint_kappa_workspace_bytes_ex(nx, ny, nz, n_src, n_rays, n_bins, step_size, c, dt, n_steps,
                                                        record_limit))


def rt_march_adjoint_kappa_ex(gbar, j, kappa, sources, n_rays, step_size, c, dt, n_steps, grad_kappa=None,
                              workspace=None, stream=None, record_limit: int = 0):
    """rt_march_adjoint_kappa with the forward-record bound of one source batch given in bytes (0 = the library's
    8 GiB): the test hook that drives the source-batch loop on small cases."""
    torch = _torch()
    _check_dev(gbar, "gbar", torch.float32, 5)
    _check_dev(j, "j", torch.float32, 4)
    _check_dev(kappa, "kappa", torch.float32, 4)
    _check_dev(sources, "sources", torch.float32, 2)
    nx, ny, nz, nb = kappa.shape
    if tuple(gbar.shape) != (n_steps, nx, ny, nz, nb) or j.shape != kappa.shape or sources.shape[1] != 3:
        raise ValueError("gbar must be [n_steps, nx, ny, nz, n_bins], j like kappa, sources [n_src, 3]")
    n_src = sources.shape[0]
    with _Call(stream, gbar, j, kappa, sources) as call:
        grad_kappa = _out_or_new(call, grad_kappa, (nx, ny, nz, nb), "grad_kappa")
        workspace = _workspace_or_new(call, workspace, rt_adjoint_kappa_workspace_bytes_ex(
            nx, ny, nz, n_src, n_rays, nb, step_size, c, dt, n_steps, record_limit))
        rc = _lib.rt_march_adjoint_kappa_ex(gbar.data_ptr(), j.data_ptr(), kappa.data_ptr(), nx, ny, nz,
                                            sources.data_ptr(), n_src, n_rays, nb, step_size, c, dt, n_steps,
                                            grad_kappa.data_ptr(), workspace.data_ptr(), workspace.numel(),
                                            call.stream_ptr, record_limit)
    if rc != RT_OK:
        raise RtError(rc, "rt_march_adjoint_kappa")
    return grad_kappa


def rt_march_adjoint_kappa(gbar, j, kappa, sources, n_rays, step_size, c, dt, n_steps, grad_kappa=None, workspace=None,
                           stream=None):
    """grad_kappa [nx,ny,nz,n_bins] = dL/dkappa for gbar [n_steps,nx,ny,nz,n_bins] = dL/d out (D19)."""
    return rt_march_adjoint_kappa_ex(gbar, j, kappa, sources, n_rays, step_size, c, dt, n_steps, grad_kappa, workspace,
                                     stream, 0)


def rt_march_single(j, kappa, source_pos, n_rays, step_size, c, dt, n_steps, out=None, workspace=None,
                    stream=None):
    torch = _torch()
    _check_dev(j, "j", torch.float32, 4)
    _check_dev(kappa, "kappa", torch.float32, 4)
    _check_dev(source_pos, "source_pos", torch.float32)
    if source_pos.numel() != 3 or kappa.shape != j.shape:
        raise ValueError("source_pos must hold 3 floats and kappa must have j's shape")
    nx, ny, nz, nb = j.shape
    with _Call(stream, j, kappa, source_pos) as call:
        out = _out_or_new(call, out, (n_steps, nx, ny, nz, nb), "out")
        workspace = _workspace_or_new(call, workspace, rt_workspace_bytes(nx, ny, nz, 1, n_rays, nb, n_steps))
        rc = _lib.rt_march_single(j.data_ptr(), kappa.data_ptr(), nx, ny, nz, source_pos.data_ptr(), n_rays, nb,
                                  step_size, c, dt, n_steps, out.data_ptr(), workspace.data_ptr(),
                                  workspace.numel(), call.stream_ptr)
    if rc != RT_OK:
        raise RtError(rc, "rt_march_single")
    return out


def rt_state_bytes(n_src: int, n_rays: int, n_bins: int) -> int:
    return int(_lib.rt_state_bytes(n_src, n_rays, n_bins))


def rt_step_workspace_bytes(nx, ny, nz, n_src, n_rays, n_bins) -> int:
    return int(_lib.rt_step_workspace_bytes(nx, ny, nz, n_src, n_rays, n_bins))


def rt_state_reset(n_src: int, n_rays: int, n_bins: int, state=None, stream=None, device=None):
    """Fresh ray state (I = 0, exp(-tau) = 1): float32 [2, n_src, n_rays, n_bins] on ``device`` (default: ``state``'s
    device, else the current CUDA device)."""
    torch = _torch()
    if state is None:
        dev = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        state = torch.empty((2, n_src, n_rays, n_bins), dtype=torch.float32, device=dev)
    _check_dev(state, "state", torch.float32)
    if state.numel() * 4 != rt_state_bytes(n_src, n_rays, n_bins):
        raise ValueError("state has the wrong size")
    with _Call(stream, state) as call:
        rc = _lib.rt_state_reset(state.data_ptr(), n_src, n_rays, n_bins, call.stream_ptr)
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
    if out is None and accumulate:
        raise ValueError("accumulate needs the running field in `out`")
    with _Call(stream, j, kappa, sources, state) as call:
        out = _out_or_new(call, out, (nx, ny, nz, nb), "out")
        workspace = _workspace_or_new(call, workspace, rt_step_workspace_bytes(nx, ny, nz, n_src, n_rays, nb))
        rc = _lib.rt_march_step(j.data_ptr(), kappa.data_ptr(), nx, ny, nz, sources.data_ptr(), n_src, n_rays, nb,
                                step_size, c, dt, int(k_begin), state.data_ptr(), out.data_ptr(),
                                int(bool(accumulate)), workspace.data_ptr(), workspace.numel(), call.stream_ptr)
    if rc != RT_OK:
        raise RtError(rc, "rt_march_step")
    return out


def _current_device(device):
    torch = _torch()
    return torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)


def rt_directions(n_rays: int, stream=None, device=None):
    torch = _torch()
    nhat = torch.empty((n_rays, 3), dtype=torch.float64, device=_current_device(device))
    with _Call(stream, nhat) as call:
        rc = _lib.rt_directions(n_rays, nhat.data_ptr(), call.stream_ptr)
    if rc != RT_OK:
        raise RtError(rc, "rt_directions")
    return nhat


def rt_ray_order(n_rays: int, stream=None, device=None):
    torch = _torch()
    order = torch.empty(rt_ray_slots(n_rays), dtype=torch.int32, device=_current_device(device))
    with _Call(stream, order) as call:
        rc = _lib.rt_ray_order(n_rays, order.data_ptr(), call.stream_ptr)
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
    with _Call(stream, j, kappa, source_pos) as call:
        pos = call.scratch((n_sub, 3), torch.float64)
        tr_i = call.scratch((n_sub, nb), torch.float32)
        tr_t = call.scratch((n_sub, nb), torch.float32)
        rc = _lib.rt_trace_ray(j.data_ptr(), kappa.data_ptr(), nx, ny, nz, nb, source_pos.data_ptr(), ray_index,
                               n_rays, step_size, n_sub, pos.data_ptr(), tr_i.data_ptr(), tr_t.data_ptr(),
                               call.stream_ptr)
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
    with _Call(stream, grid) as call:
        rc = _lib.rt_bench_red_ceiling(mode, grid.data_ptr(), nx, ny, nz, nb, n_red, seed, ctypes.byref(issued),
                                       call.stream_ptr)
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
