"""N > 1 is "replicas only": every rank renders the same trajectory on its own GPU and the only
cross-rank step is the max over ranks of the device time (bench.py).  That step is covered here with two gloo
processes on the CPU; there is no data-path collective to test."""
import os
import sys

import pytest
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms_local = 10.0 + 5.0 * rank                       # rank 1 is the slow one
    ms = bench.max_over_ranks(ms_local, world)
    dist.barrier()
    q.put((rank, ms, bench.aggregate_fps(world, 300, ms)))
    dist.destroy_process_group()


def test_max_over_ranks_and_weak_scaling_value():
    world, port = 2, 29500 + os.getpid() % 2000
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, fps in out:
        assert ms == pytest.approx(15.0)               # every rank sees the slowest rank's time
        assert fps == pytest.approx(2 * 300 / 15e-3)   # frames of all replicas over that time


def test_single_rank_is_identity():
    import bench
    assert bench.max_over_ranks(7.5, 1) == 7.5
    assert bench.aggregate_fps(1, 300, 200.0) == pytest.approx(1500.0)
