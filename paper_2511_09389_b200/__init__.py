"""B200-native ray march of Ray-trax (arXiv 2511.09389): hand-written sm_100a CUDA behind a C ABI.

``include/rtmarch.h`` is the boundary; ``binding`` marshals arguments to it; ``sharding`` is the multi-GPU plumbing.
The binding (and with it ``librtmarch.so``) is loaded on the first use of one of its names, not when the package is
imported: ``import paper_2511_09389_b200.sharding`` alone maps no native code.  Loading raises if the library is
missing and cannot be built: there is no CPU fallback.
"""
import importlib

_BINDING_NAMES = (
    "RT_EALIGN", "RT_ECUDA", "RT_EINVAL", "RT_ETOOBIG", "RT_EWORKSPACE", "RT_OK", "RT_VARIANT_DEFAULT", "RT_VARIANT_DIRECT",
    "RT_VARIANT_DIRECT_COHERENT", "RT_VARIANT_FLAG_ACC_F32", "RT_VARIANT_FLAG_ONE_BIN", "RT_VARIANT_SLIDING_BY_DIRECTION",
    "RT_VARIANT_SLIDING_BY_SOURCE", "RT_VARIANT_SLIDING_LATTICE", "RtError", "alloc_workspace", "library_path",
    "rt_bench_red_ceiling", "rt_directions", "rt_host_release", "rt_launch_count", "rt_adjoint_kappa_workspace_bytes",
    "rt_adjoint_kappa_workspace_bytes_ex", "rt_adjoint_workspace_bytes", "rt_march", "rt_march_adjoint_j",
    "rt_march_adjoint_kappa", "rt_march_adjoint_kappa_ex", "rt_march_ex", "rt_march_jvp_kappa", "rt_march_host", "rt_march_single",
    "rt_march_step", "rt_march_trilinear_kappa", "rt_state_bytes", "rt_state_reset", "rt_step_workspace_bytes",
    "rt_ray_order", "rt_ray_slots", "rt_strerror", "rt_substeps_per_step", "rt_trace_ray", "rt_version",
    "rt_workspace_bytes", "rt_march_static", "rt_static_workspace_bytes")

__all__ = list(_BINDING_NAMES) + ["binding", "sharding", "build"]


def __getattr__(name):
    if name in _BINDING_NAMES:
        return getattr(importlib.import_module(".binding", __name__), name)
    if name in ("binding", "sharding", "build"):
        return importlib.import_module("." + name, __name__)
    raise AttributeError(f"module {__name__!r} has no attribute {name!r}")
