"""Worker of the two-rank tests in test_gpu_sharded.py: one process per rank, each with its own plan and its own
shard of the particles, running Plan.energy_forces_sharded through a real torch.distributed collective."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def case_inputs(case: str):
    """(r, q, plan keyword arguments) of a named case; the same on every rank and in the parent test."""
    from enuf_inputs import make_workload, random_neutral_gas
    if case == "cfg1":
        w = make_workload("cfg1")
        return w.r, w.q, dict(L=w.L, alpha=w.alpha, k_cut=w.k_cut, M=w.M, sigma=w.sigma, m=w.m, window=w.window,
                              dtype="f64")
    if case == "gas20k":
        N, L = 20000, 30.0
        r, q = random_neutral_gas(N, L, seed=7, dtype=np.float32)
        return r, q, dict(L=L, alpha=0.9, k_cut=16, M=32, sigma=2.0, m=6, window="kaiser_bessel", dtype="f32")
    raise ValueError(case)


def run(rank: int, world: int, backend: str, port: int, case: str, outdir: str) -> None:
    import torch
    import torch.distributed as dist
    import paper_2004_12484_b200 as enuf

    dev = rank % torch.cuda.device_count()          # gloo variant: both ranks may share cuda:0
    torch.cuda.set_device(dev)
    kw = dict(backend=backend, init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    if backend == "nccl":
        kw["device_id"] = torch.device("cuda", dev)
    dist.init_process_group(**kw)
    try:
        r, q, pk = case_inputs(case)
        lo, hi = enuf.shard_bounds(q.shape[0], rank, world)
        tdt = torch.float64 if pk["dtype"] == "f64" else torch.float32
        plan = enuf.Plan(hi - lo, pk["L"], pk["alpha"], pk["k_cut"], pk["M"], sigma=pk["sigma"], m=pk["m"],
                         dtype=tdt, window=pk["window"])
        rt = torch.from_numpy(np.ascontiguousarray(r[lo:hi])).cuda()
        qt = torch.from_numpy(np.ascontiguousarray(q[lo:hi])).cuda()
        for _ in range(2):                            # twice: the second call reuses every buffer
            E, F = plan.energy_forces_sharded(rt, qt)
        np.savez(os.path.join(outdir, f"rank{rank}.npz"), E=E, F=F.cpu().numpy().astype(np.float64), lo=lo, hi=hi)
        plan.close()
        dist.barrier()
    finally:
        dist.destroy_process_group()


if __name__ == "__main__":
    run(int(sys.argv[1]), int(sys.argv[2]), sys.argv[3], int(sys.argv[4]), sys.argv[5], sys.argv[6])
