"""CPU-only, world_size-2 (gloo) check of bench.py's multi-GPU bookkeeping.  The path has no exchange step
("replicas only"): N ranks run N independent replicas, the step time is the max over ranks and the
value is the sum of the replicas' work over that time.  No compute runs here."""
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
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, dist, torch.device("cpu"))      # rank 1 is the slow one
    q.put((rank, ms, bench.replicas_value(world, 2.0e12, ms)))
    dist.destroy_process_group()


def test_two_replicas_take_the_max_time_and_sum_the_work():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 1000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, value in res:
        assert ms == 15.0                                   # max over ranks, on every rank
        assert abs(value - 2 * 2.0e12 / 15e-3 / 1e12) < 1e-9   # whole-job aggregate of two replicas


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(7.5, None, torch.device("cpu")) == 7.5
    assert abs(bench.replicas_value(1, 1.0e12, 1000.0) - 1.0) < 1e-12
