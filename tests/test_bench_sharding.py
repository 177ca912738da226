"""bench.py's N>1 path on CPU: beam sharding with no exchange step, timing = max over ranks (gloo, world_size 2)."""
import os
import sys

import pytest
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms_rank = 10.0 + 5.0 * rank                       # rank 1 is the slow one
    value, ms = bench.job_throughput(1000.0, world, ms_rank)
    mx = bench.max_over_ranks(float(rank), world)
    dist.barrier()
    q.put((rank, value, ms, mx))
    dist.destroy_process_group()


def test_job_throughput_world2_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    for rank, value, ms, mx in res:
        assert ms == pytest.approx(15.0)              # the slowest rank's time, on every rank
        assert value == pytest.approx(2 * 1000.0 / 15e-3)   # units of all ranks / that time
        assert mx == 1.0


def test_job_throughput_single_rank_identity():
    sys.path.insert(0, ROOT)
    import bench
    v, ms = bench.job_throughput(500.0, 1, 4.0)
    assert ms == 4.0 and v == pytest.approx(500.0 / 4e-3)
