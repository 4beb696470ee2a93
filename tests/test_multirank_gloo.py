"""N > 1 host logic on CPU: two gloo ranks on 127.0.0.1.

  - bench.py's replica mode: max-over-ranks time, sum of launches / particles;
  - the sharded path's host side: contiguous particle shards (shard_bounds) and the one exchange
    step, an all-reduce (sum) of the partial spectra (all_reduce_sum_), checked through Eq. 61
    (PAPER.md:533-540): the direct structure factors of the two shards, summed over the gloo
    group by the SAME helper the GPU path calls, equal the structure factor of the whole system."""
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


def _shard_worker(rank: int, world: int, port: int, out):
    import numpy as np
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import paper_2004_12484_b200 as enuf
    from enuf_inputs import make_workload
    from oracle import enuf_oracle as O
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = make_workload("cfg1")
    ml = O.modes(w.k_cut)[:200]
    lo, hi = enuf.shard_bounds(w.N - 1, rank, world)            # 999 particles: uneven shards
    S_part = O.direct_S(w.r[lo:hi], w.q[lo:hi], w.L, ml)
    buf = torch.from_numpy(np.ascontiguousarray(np.stack([S_part.real, S_part.imag], axis=1)))
    enuf.all_reduce_sum_(buf)
    S_full = O.direct_S(w.r[:w.N - 1], w.q[:w.N - 1], w.L, ml)
    err = float(np.abs(buf.numpy()[:, 0] + 1j * buf.numpy()[:, 1] - S_full).max() / np.abs(S_full).max())
    out.put((rank, lo, hi, err))
    dist.destroy_process_group()


def test_two_gloo_ranks_shard_and_sum_partial_structure_factors(oracle):
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_shard_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [(lo, hi) for _, lo, hi, _ in res] == [(0, 500), (500, 999)]
    for _, _, _, err in res:
        assert err <= 1e-13


def test_shard_bounds_partition():
    sys.path.insert(0, ROOT)
    import paper_2004_12484_b200 as enuf
    for N in (0, 1, 7, 1000, 1_000_003):
        for world in (1, 2, 3, 8):
            b = [enuf.shard_bounds(N, r, world) for r in range(world)]
            assert b[0][0] == 0 and b[-1][1] == N
            assert all(b[i][1] == b[i + 1][0] for i in range(world - 1))
            sizes = [hi - lo for lo, hi in b]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        enuf.shard_bounds(10, 2, 2)
