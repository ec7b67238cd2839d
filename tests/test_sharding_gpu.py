"""The N > 1 path on devices: two NCCL ranks, one per GPU, each marching its slice of
the sources with the real rt_march, one sum all-reduce of the field, compared with the fp64 oracle on all sources.
Needs two GPUs in the box; skipped (with the reason) on a one-GPU box."""
import os
import socket
import sys

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
torch = pytest.importorskip("torch")


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.setdefault("NCCL_DEBUG", "WARN")
    import torch.distributed as dist

    import paper_2511_09389_b200 as rt
    import workloads
    from paper_2511_09389_b200 import sharding
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world,
                            device_id=torch.device("cuda", rank))
    w = workloads.make_config("C1")
    dev = torch.device("cuda", rank)
    j, k = torch.from_numpy(w.j).to(dev), torch.from_numpy(w.kappa).to(dev)
    src = torch.from_numpy(w.sources).to(dev)

    def march_fn(j, k, s, *a):
        return rt.rt_march(j, k, s.contiguous(), *a)

    field = sharding.sharded_march(march_fn, j, k, src, w.n_rays, w.step_size, w.c, w.dt, w.n_steps, rank=rank,
                                   world_size=world,
                                   zeros_fn=lambda: torch.zeros((w.n_steps,) + w.j.shape, dtype=torch.float32, device=dev))
    torch.cuda.synchronize()
    q.put((rank, field.cpu().numpy()))
    dist.barrier()
    dist.destroy_process_group()


def test_two_nccl_ranks_match_the_oracle(oracle_mod):
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device")
    if torch.cuda.device_count() < 2:
        pytest.skip(f"needs 2 GPUs for 2 NCCL ranks; this box has {torch.cuda.device_count()} "
                    "(the host logic runs on CPU in tests/test_sharding_cpu.py)")
    import torch.multiprocessing as mp

    import parity
    import workloads
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = dict(q.get(timeout=300) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    w = workloads.make_config("C1")
    ref = oracle_mod.march(w.j, w.kappa, w.sources, w.n_rays, w.step_size, w.c, w.dt, w.n_steps)
    for r in range(2):
        parity.assert_parity(got[r], ref, f"2 NCCL ranks, rank {r}")
    assert np.array_equal(got[0], got[1])          # the all-reduce leaves the same bits on every rank
