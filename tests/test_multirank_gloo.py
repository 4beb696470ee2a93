"""N > 1 plumbing of bench.py on CPU: two gloo ranks (replicas only).

The path has no data-path collective; what the N-GPU run adds is the max-over-ranks time and
the sum of launches / particles.  These are exercised here with world_size 2 on 127.0.0.1."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    t_rank = 1.5 + rank                                  # rank 1 is the slow one
    t_max = bench.reduce_over_ranks(t_rank, "max", "cpu")
    launches = bench.reduce_over_ranks(12.0 * (rank + 1), "sum", "cpu")
    dist.barrier()
    out.put((rank, t_max, launches, bench.whole_job_value(1000, world, t_max)))
    dist.destroy_process_group()


def test_two_gloo_ranks_reduce_time_and_counts():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, t_max, launches, value in res:
        assert t_max == 2.5                               # max over ranks, identical on both
        assert launches == 36.0                           # sum over ranks
        assert value == pytest.approx(2 * 1000 / 2.5e-3)  # all ranks' particles / slowest time


def test_single_process_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_over_ranks(3.25, "max", "cpu") == 3.25
    assert bench.whole_job_value(10, 1, 2.0) == pytest.approx(5000.0)
