"""The N > 1 path of bench.py on CPU: two gloo ranks.  The path is "replicas only" (north_star: one GPU
per problem, no sharding, no data-path collective), so what there is to test is the contract's
aggregation: device times reduced with MAX over ranks, value = work of ALL ranks / that time, and that
only rank 0 would print."""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        mine = [0.010 * (rank + 1), 0.5 - 0.1 * rank, 0.02]          # rank-dependent "seconds"
        got = bench.max_over_ranks(mine, torch.device("cpu"), world)
        dist.barrier()
        q.put((rank, got, bench.aggregate_gflops(3.0e9, 20, got[0], world)))
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_max_over_ranks_and_aggregate():
    import torch.multiprocessing as mp
    world, port = 2, 29731
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, got, gf in res:
        assert got == pytest.approx([0.020, 0.5, 0.02])                 # max over the two ranks
        assert gf == pytest.approx(2 * 3.0e9 * 20 / 0.020 * 1e-9)        # both replicas' work / max time


def test_single_rank_is_identity():
    import torch
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([1.5, 2.5], torch.device("cpu"), 1) == [1.5, 2.5]
    assert bench.aggregate_gflops(1e9, 10, 0.5, 1) == pytest.approx(20.0)
