"""The N > 1 path on CPU: world_size-2 gloo process group, sources sharded, one sum all-reduce of the field.
The per-rank march is stood in for by the oracle (test infrastructure) — what is under test is the host
logic of paper_2511_09389_b200/sharding.py: the partition covers every source once and the reduced field
equals the unsharded field (the field is a sum over sources)."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
torch = pytest.importorskip("torch")


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _problem(n_src):
    rng = np.random.default_rng(11)
    j = rng.uniform(0.1, 1.0, (6, 5, 7, 2)).astype(np.float32)
    k = rng.uniform(0.0, 0.5, (6, 5, 7, 2)).astype(np.float32)
    src = rng.uniform(-1.0, 7.0, (n_src, 3)).astype(np.float32)
    return j, k, src


def _worker(rank, world, port, n_src, q):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist

    import oracle
    from paper_2511_09389_b200 import sharding
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    j, k, src = _problem(n_src)

    def march_fn(j, k, s, *a):
        return torch.from_numpy(oracle.march(j, k, s, *a, n_threads=1))

    field = sharding.sharded_march(march_fn, j, k, src, 12, 0.5, 1.0, 3.0, 2, rank=rank, world_size=world,
                                   zeros_fn=lambda: torch.zeros((2, 6, 5, 7, 2), dtype=torch.float64))
    q.put((rank, field.numpy()))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("n_src", [5, 1])
def test_two_ranks_reduce_to_the_unsharded_field(n_src):
    import torch.multiprocessing as mp

    import oracle
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, n_src, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = dict(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    j, k, src = _problem(n_src)
    want = oracle.march(j, k, src, 12, 0.5, 1.0, 3.0, 2, n_threads=1)
    for r in range(2):
        np.testing.assert_allclose(got[r], want, rtol=1e-13, atol=0)


def test_source_slices_partition_the_sources():
    from paper_2511_09389_b200.sharding import source_slice
    for n in (0, 1, 7, 2097, 16776):
        for world in (1, 2, 3, 8):
            seen = np.zeros(n, dtype=int)
            sizes = []
            for r in range(world):
                sl = source_slice(n, r, world)
                seen[sl] += 1
                sizes.append(sl.stop - sl.start)
            assert (seen == 1).all() and max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        source_slice(4, 2, 2)


def test_bench_weak_scaling_workload_extends_the_source_list():
    """bench.py --gpus N: rank r marches the r-th block of N * n_src sources placed by the config's own rule."""
    sys.path.insert(0, ROOT)
    import bench
    from paper_2511_09389_b200.sharding import source_slice
    one = bench.make_workload("C1", 1)
    two = bench.make_workload("C1", 2)
    assert two.n_src == 2 * one.n_src and two.sources.dtype == np.float32
    assert np.array_equal(two.j, one.j) and np.array_equal(two.kappa, one.kappa)
    blocks = [two.sources[source_slice(two.n_src, r, 2)] for r in range(2)]
    assert all(len(b) == one.n_src for b in blocks)
    assert len(np.unique(np.concatenate(blocks), axis=0)) == two.n_src          # disjoint, all distinct
    desc = bench.describe(one, 2)
    assert "2 GPU" in desc["parallelism"] and desc["updates_per_gpu"] == one.updates
