"""N > 1 host logic on CPU (gloo, world_size 2): the path does not shard across GPUs (DESIGN.md "Multi-GPU":
replicas only), so the only collective of a multi-GPU bench run is the MAX of the per-rank step times."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms, e2e = bench.max_over_ranks([2.0 + rank, 5.0 - rank], dist, torch.device("cpu"))
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, ms, e2e, bench.aggregate_value(4096, world, ms)))


def test_max_over_ranks_and_aggregate_value_gloo():
    world, port = 2, 29500 + os.getpid() % 2000
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, e2e, value in res:
        assert ms == 3.0 and e2e == 5.0                    # the slowest rank decides, on every rank
        assert value == 2 * 4096 / 3.0e-3                  # whole-job aggregate of two replicas


def test_single_rank_passthrough():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([1.5, 2.5], None, None) == [1.5, 2.5]
    assert bench.aggregate_value(4096, 1, 2.0) == 4096 / 2.0e-3
