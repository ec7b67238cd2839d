"""ctypes loader for the fp64 CPU oracle (``oracle/rt_oracle.cpp``).  TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It imports nothing from ``paper_2511_09389_b200`` and the CUDA path imports
nothing from here.  ``build()`` compiles the single C++ file with g++; nothing else is needed.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rt_oracle.cpp")
_LIB = os.path.join(_HERE, "librtoracle.so")
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """Compile ``rt_oracle.cpp`` -> ``librtoracle.so`` (plain g++ -O2, no fast-math, no contraction)."""
    if (not force and os.path.exists(_LIB) and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    tmp = _LIB + f".tmp{os.getpid()}"
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-pthread", "-Wall", "-Wextra",
           "-o", tmp, _SRC]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _LIB)
    return _LIB


def lib() -> ctypes.CDLL:
    global _lib
    with _lock:
        if _lib is None:
            L = ctypes.CDLL(build())
            fp = ctypes.POINTER(ctypes.c_float)
            dp = ctypes.POINTER(ctypes.c_double)
            L.rt_oracle_substeps.restype = ctypes.c_long
            L.rt_oracle_substeps.argtypes = [ctypes.c_float] * 3
            L.rt_oracle_direction.restype = ctypes.c_int
            L.rt_oracle_direction.argtypes = [ctypes.c_long, ctypes.c_long, dp]
            L.rt_oracle_trace_ray.restype = ctypes.c_int
            L.rt_oracle_trace_ray.argtypes = [fp, fp, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, fp,
                                              ctypes.c_long, ctypes.c_long, ctypes.c_float, ctypes.c_long,
                                              dp, dp, dp, dp]
            L.rt_march_oracle.restype = ctypes.c_int
            L.rt_march_oracle.argtypes = [fp, fp, ctypes.c_int, ctypes.c_int, ctypes.c_int, fp, ctypes.c_int,
                                          ctypes.c_int, ctypes.c_int, ctypes.c_float, ctypes.c_float,
                                          ctypes.c_float, ctypes.c_int, dp, ctypes.c_int]
            L.rt_oracle_trace_ray_k.restype = ctypes.c_int
            L.rt_oracle_trace_ray_k.argtypes = L.rt_oracle_trace_ray.argtypes + [ctypes.c_int]
            L.rt_march_oracle_k.restype = ctypes.c_int
            L.rt_march_oracle_k.argtypes = L.rt_march_oracle.argtypes + [ctypes.c_int]
            L.rt_adjoint_j_oracle.restype = ctypes.c_int
            L.rt_adjoint_j_oracle.argtypes = [dp, fp, ctypes.c_int, ctypes.c_int, ctypes.c_int, fp, ctypes.c_int,
                                              ctypes.c_int, ctypes.c_int, ctypes.c_float, ctypes.c_float,
                                              ctypes.c_float, ctypes.c_int, dp, ctypes.c_int]
            L.rt_adjoint_kappa_oracle.restype = ctypes.c_int
            L.rt_adjoint_kappa_oracle.argtypes = [dp, fp, fp, ctypes.c_int, ctypes.c_int, ctypes.c_int, fp, ctypes.c_int,
                                                  ctypes.c_int, ctypes.c_int, ctypes.c_float, ctypes.c_float,
                                                  ctypes.c_float, ctypes.c_int, dp, ctypes.c_int]
            L.rt_jvp_kappa_oracle.restype = ctypes.c_int
            L.rt_jvp_kappa_oracle.argtypes = [fp, fp, fp, ctypes.c_int, ctypes.c_int, ctypes.c_int, fp, ctypes.c_int,
                                              ctypes.c_int, ctypes.c_int, ctypes.c_float, ctypes.c_float, ctypes.c_float,
                                              ctypes.c_int, dp, ctypes.c_int]
            L.rt_oracle_step.restype = ctypes.c_int
            L.rt_oracle_step.argtypes = [fp, fp, ctypes.c_int, ctypes.c_int, ctypes.c_int, fp, ctypes.c_int,
                                         ctypes.c_int, ctypes.c_int, ctypes.c_float, ctypes.c_float, ctypes.c_float,
                                         ctypes.c_long, dp, dp, ctypes.c_int]
            L.rt_oracle_version.restype = ctypes.c_char_p
            _lib = L
    return _lib


def _f32(a, ndim):
    a = np.ascontiguousarray(a, dtype=np.float32)
    if a.ndim != ndim:
        raise ValueError(f"expected {ndim}-d array, got shape {a.shape}")
    return a


def _fp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_float))


def _dp(a):
    return None if a is None else a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def host_threads() -> int:
    """Cores this process may run on (the oracle's default thread count)."""
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:  # pragma: no cover
        return os.cpu_count() or 1


def substeps(step_size: float, c: float, dt: float) -> int:
    return int(lib().rt_oracle_substeps(step_size, c, dt))


def direction(i: int, n: int) -> np.ndarray:
    out = np.zeros(3)
    if lib().rt_oracle_direction(i, n, _dp(out)):
        raise ValueError("bad direction index")
    return out


def march(j, kappa, sources, n_rays, step_size, c, dt, n_steps, n_threads: int | None = None,
          max_private_bytes: int = 24 << 30, kappa_trilinear: bool = False) -> np.ndarray:
    """Oracle field: float64 ``[n_steps, nx, ny, nz, n_bins]`` (cumulative snapshots, scaled by 4π/N_Ω)."""
    j = _f32(j, 4)
    kappa = _f32(kappa, 4)
    sources = _f32(sources, 2)
    if kappa.shape != j.shape or sources.shape[1] != 3:
        raise ValueError("shape mismatch")
    nx, ny, nz, nb = j.shape
    if n_threads is None:
        n_threads = host_threads()
    # each thread owns one private fp64 grid: bound the total
    n_threads = max(1, min(n_threads, max_private_bytes // max(1, j.size * 8)))
    out = np.empty((n_steps, nx, ny, nz, nb), dtype=np.float64)
    rc = lib().rt_march_oracle_k(_fp(j), _fp(kappa), nx, ny, nz, _fp(sources), sources.shape[0], n_rays, nb,
                                 step_size, c, dt, n_steps, _dp(out), n_threads, int(kappa_trilinear))
    if rc:
        raise ValueError("rt_march_oracle: invalid arguments")
    return out


def adjoint_j(gbar, kappa, sources, n_rays, step_size, c, dt, n_steps, n_threads: int | None = None) -> np.ndarray:
    """dL/dj for dL/d out[m] = gbar[m]: float64 [nx, ny, nz, n_bins] (the march is linear in j; D19)."""
    kappa = _f32(kappa, 4)
    sources = _f32(sources, 2)
    nx, ny, nz, nb = kappa.shape
    gbar = np.ascontiguousarray(gbar, dtype=np.float64)
    if gbar.shape != (n_steps, nx, ny, nz, nb):
        raise ValueError("gbar must be [n_steps, nx, ny, nz, n_bins]")
    if n_threads is None:
        n_threads = host_threads()
    n_threads = max(1, min(n_threads, (24 << 30) // max(1, kappa.size * 8)))
    grad = np.empty((nx, ny, nz, nb), dtype=np.float64)
    rc = lib().rt_adjoint_j_oracle(_dp(gbar), _fp(kappa), nx, ny, nz, _fp(sources), sources.shape[0], n_rays, nb,
                                   step_size, c, dt, n_steps, _dp(grad), n_threads)
    if rc:
        raise ValueError("rt_adjoint_j_oracle: invalid arguments")
    return grad


def adjoint_kappa(gbar, j, kappa, sources, n_rays, step_size, c, dt, n_steps, n_threads: int | None = None) -> np.ndarray:
    """dL/dkappa for dL/d out[m] = gbar[m]: float64 [nx, ny, nz, n_bins] (D19)."""
    j = _f32(j, 4)
    kappa = _f32(kappa, 4)
    sources = _f32(sources, 2)
    nx, ny, nz, nb = kappa.shape
    gbar = np.ascontiguousarray(gbar, dtype=np.float64)
    if gbar.shape != (n_steps, nx, ny, nz, nb) or j.shape != kappa.shape:
        raise ValueError("gbar must be [n_steps, nx, ny, nz, n_bins] and j must have kappa's shape")
    if n_threads is None:
        n_threads = host_threads()
    n_threads = max(1, min(n_threads, (24 << 30) // max(1, kappa.size * 8)))
    grad = np.empty((nx, ny, nz, nb), dtype=np.float64)
    rc = lib().rt_adjoint_kappa_oracle(_dp(gbar), _fp(j), _fp(kappa), nx, ny, nz, _fp(sources), sources.shape[0], n_rays,
                                       nb, step_size, c, dt, n_steps, _dp(grad), n_threads)
    if rc:
        raise ValueError("rt_adjoint_kappa_oracle: invalid arguments")
    return grad


def jvp_kappa(j, kappa, dkappa, sources, n_rays, step_size, c, dt, n_steps, n_threads: int | None = None) -> np.ndarray:
    """Tangent of the field for kappa -> kappa + eps * dkappa at eps = 0 (D21): float64
    [n_steps, nx, ny, nz, n_bins], cumulative snapshots like ``march``."""
    j = _f32(j, 4)
    kappa = _f32(kappa, 4)
    dkappa = _f32(dkappa, 4)
    sources = _f32(sources, 2)
    if kappa.shape != j.shape or dkappa.shape != j.shape or sources.shape[1] != 3:
        raise ValueError("shape mismatch")
    nx, ny, nz, nb = j.shape
    if n_threads is None:
        n_threads = host_threads()
    n_threads = max(1, min(n_threads, (24 << 30) // max(1, j.size * 8 * n_steps)))
    out = np.empty((n_steps, nx, ny, nz, nb), dtype=np.float64)
    rc = lib().rt_jvp_kappa_oracle(_fp(j), _fp(kappa), _fp(dkappa), nx, ny, nz, _fp(sources), sources.shape[0], n_rays, nb,
                                   step_size, c, dt, n_steps, _dp(out), n_threads)
    if rc:
        raise ValueError("rt_jvp_kappa_oracle: invalid arguments")
    return out


def new_state(n_src: int, n_rays: int, n_bins: int) -> np.ndarray:
    """Fresh ray state for ``step``: float64 [n_src, n_rays, 2, n_bins] = (I, tau), all zero (I_0 = tau_0 = 0)."""
    return np.zeros((n_src, n_rays, 2, n_bins), dtype=np.float64)


def step(j, kappa, sources, n_rays, step_size, c, dt, k_begin: int, state: np.ndarray,
         n_threads: int | None = None) -> np.ndarray:
    """One time step in the given medium from substep ``k_begin``; updates ``state`` in place and returns the
    increment of the field, float64 [nx, ny, nz, n_bins] (scaled by 4π/N_Ω)."""
    j = _f32(j, 4)
    kappa = _f32(kappa, 4)
    sources = _f32(sources, 2)
    nx, ny, nz, nb = j.shape
    if state.dtype != np.float64 or not state.flags.c_contiguous or state.shape != (sources.shape[0], n_rays, 2, nb):
        raise ValueError("state must be the C-contiguous float64 array of new_state()")
    if n_threads is None:
        n_threads = host_threads()
    n_threads = max(1, min(n_threads, (24 << 30) // max(1, j.size * 8)))
    inc = np.empty((nx, ny, nz, nb), dtype=np.float64)
    rc = lib().rt_oracle_step(_fp(j), _fp(kappa), nx, ny, nz, _fp(sources), sources.shape[0], n_rays, nb, step_size,
                              c, dt, k_begin, _dp(state), _dp(inc), n_threads)
    if rc:
        raise ValueError("rt_oracle_step: invalid arguments")
    return inc


def trace_ray(j, kappa, source_pos, ray_index, n_rays, step_size, n_sub, deposit: bool = False,
              kappa_trilinear: bool = False):
    """One ray from k=0: returns dict(I=[n_sub,B], tau=[n_sub,B], pos=[n_sub,3], acc=unnormalised grid|None)."""
    j = _f32(j, 4)
    kappa = _f32(kappa, 4)
    src = _f32(np.asarray(source_pos).reshape(3), 1)
    nx, ny, nz, nb = j.shape
    I = np.zeros((n_sub, nb))
    tau = np.zeros((n_sub, nb))
    pos = np.zeros((n_sub, 3))
    acc = np.zeros((nx, ny, nz, nb)) if deposit else None
    rc = lib().rt_oracle_trace_ray_k(_fp(j), _fp(kappa), nx, ny, nz, nb, _fp(src), ray_index, n_rays, step_size,
                                     n_sub, _dp(I), _dp(tau), _dp(pos), _dp(acc), int(kappa_trilinear))
    if rc:
        raise ValueError("rt_oracle_trace_ray: invalid arguments")
    return {"I": I, "tau": tau, "pos": pos, "acc": acc}
