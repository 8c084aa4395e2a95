"""The N > 1 path of bench.py is "replicas only": no data-path collective, only the timing reduction
(max over ranks) and the whole-job aggregation.  Exercised here with world_size 2 on the gloo backend (CPU)."""
import os
import sys

import pytest
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
    try:
        my_ms = 3.0 + rank                       # rank 1 is the slow one
        t = bench.max_over_ranks(my_ms, dist, torch.device("cpu"))
        dist.barrier()
        v = bench.job_throughput(world, 1000, t * 1e-3)
        q.put((rank, t, v))
    finally:
        dist.destroy_process_group()


def test_replica_aggregation_world_size_2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 1000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, t, v in res:
        assert t == 4.0                          # max over ranks, seen identically by both
        assert v == pytest.approx(2 * 1000 / 4.0e-3)


def test_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(2.5, None, None) == 2.5
    assert bench.job_throughput(1, 10, 2.0) == 5.0


def test_reference_arm_non_zero_ranks_do_no_work(monkeypatch):
    sys.path.insert(0, ROOT)
    import bench

    class A:
        config, steps, warmup, gpus = 5, 1, 0, 2
    monkeypatch.setenv("RANK", "1")
    assert bench.run_reference(A()) == 0         # returns at once, prints nothing
