"""Multi-GPU plumbing: the march shards over SOURCES (rays are independent given the medium, PAPER.md:33;
the field is a plain sum over sources).  j and kappa are replicated, each rank marches its own
contiguous slice of the sources into a private field, and ONE sum all-reduce of the field
(n_steps * N_cells * n_bins floats) over torch.distributed (NCCL on GPUs, gloo in the CPU tests) gives every
rank the total — the B200 counterpart of the paper's "final on-device sum per shard before reducing across
shards", without its N_Omega % n_dev == 0 restriction.  No arithmetic of the method lives here.
"""
from __future__ import annotations


def source_slice(n_src: int, rank: int, world_size: int) -> slice:
    """Contiguous, balanced partition of range(n_src): sizes differ by at most one, empty slices allowed."""
    if world_size < 1 or not (0 <= rank < world_size) or n_src < 0:
        raise ValueError("bad rank/world_size/n_src")
    lo = n_src * rank // world_size
    hi = n_src * (rank + 1) // world_size
    return slice(lo, hi)


def allreduce_field(field, group=None):
    """In-place sum of the per-rank fields (torch tensor) over the process group; returns the tensor."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(field, op=dist.ReduceOp.SUM, group=group)
    return field


def sharded_march(march_fn, j, kappa, sources, *args, rank: int, world_size: int, zeros_fn, group=None, **kw):
    """march_fn(j, kappa, sources_shard, *args, **kw) on this rank's slice, then the all-reduce.

    ``zeros_fn()`` supplies the zero field for a rank whose slice is empty (n_src < world_size)."""
    sl = source_slice(int(sources.shape[0]), rank, world_size)
    mine = sources[sl]
    field = march_fn(j, kappa, mine, *args, **kw) if mine.shape[0] > 0 else zeros_fn()
    return allreduce_field(field, group)
