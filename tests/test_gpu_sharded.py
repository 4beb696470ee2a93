"""Sharded (multi-GPU) evaluation on ONE GPU: the two C-ABI halves with the all-reduce done by hand.

HP-ENUF: every rank spreads and forward-transforms its own particles, the partial
spectra are summed over ranks (Eq. 61, :533-540), and every rank finishes (scale, energy, inverse
transform, gather onto its own particles).  Here the "ranks" are plans on the same device and the sum
is a tensor add of the plans' spectrum buffers, so the arithmetic of the N-GPU path is exercised
exactly.  The collective is exercised by the two-rank tests at the end: two processes, one plan and one
shard each, Plan.energy_forces_sharded through torch.distributed -- over gloo with both ranks on cuda:0
(runs on a one-GPU box) and over NCCL when the box has two GPUs (skipped otherwise).  The one-rank NCCL
test only checks the call sequence (with one rank all_reduce_sum_ returns before the collective).
"""
import math
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

from enuf_inputs import make_workload, random_neutral_gas

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def enuf(torch_cuda):
    import paper_2004_12484_b200 as e
    e.lib()
    return e


def rel_rms(a, b):
    a = np.asarray(a, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    return math.sqrt(((a - b) ** 2).sum() / max((b ** 2).sum(), 1e-300))


def sharded_eval(enuf, torch, r, q, world, make_plan):
    """Evaluate with `world` plans, one per contiguous shard; returns (E per rank, F of the whole system)."""
    N = q.shape[0]
    plans, parts = [], []
    for rank in range(world):
        lo, hi = enuf.shard_bounds(N, rank, world)
        plan = make_plan(hi - lo)
        rt = torch.from_numpy(np.ascontiguousarray(r[lo:hi])).cuda()
        qt = torch.from_numpy(np.ascontiguousarray(q[lo:hi])).cuda()
        Ft = torch.empty((hi - lo, 3), dtype=rt.dtype, device="cuda")
        plan.spectrum_partial(rt, qt, Ft)
        plans.append(plan); parts.append((rt, qt, Ft))
    total = torch.zeros_like(plans[0].spectrum_tensor())
    for plan in plans:                                   # the all-reduce (sum), rank order
        total += plan.spectrum_tensor()
    Es, Fs = [], []
    for plan, (rt, qt, Ft) in zip(plans, parts):
        plan.spectrum_tensor().copy_(total)
        E, F = plan.forces_from_spectrum(Ft)
        Es.append(E); Fs.append(F.cpu().numpy())
        plan.close()
    return Es, np.concatenate(Fs, axis=0)


@pytest.mark.parametrize("name,variant,world", [("cfg1", "analytic", 2), ("cfg1", "ik", 3), ("cfg2", "analytic", 4)])
def test_sharded_fp64_matches_oracle_b(enuf, torch_cuda, oracle, name, variant, world):
    torch = torch_cuda
    w = make_workload(name)
    ref = oracle.enuf_workload(w, variant=variant)
    Es, F = sharded_eval(enuf, torch, w.r, w.q, world,
                         lambda n: enuf.Plan(n, w.L, w.alpha, w.k_cut, w.M, sigma=w.sigma, m=w.m,
                                             dtype=torch.float64, window=w.window, variant=variant,
                                             slater_lambda=w.slater_lambda))
    assert all(E == Es[0] for E in Es)                    # same summed bytes, fixed-order reduction
    assert abs(Es[0] - ref["E"]) <= 1e-12 * abs(ref["E"])
    assert rel_rms(F, ref["F"]) <= 1e-11


@pytest.mark.parametrize("variant,world", [("analytic", 2), ("ik", 3)])
def test_sharded_on_a_grid_of_three_times_a_power_of_two(enuf, torch_cuda, oracle, variant, world):
    """sigma_s = 1.5 (M = 32 on the 48^3 grid, the mixed-radix FFT path): the buffer the ranks exchange is the full complex
    spectrum after the three forward passes; Eq. 61 holds for it just the same."""
    torch = torch_cuda
    N, L, n, M, m = 1200, 8.0, 48, 32, 4
    r, q = random_neutral_gas(N, L, seed=48)
    k_cut, alpha = M // 2, 1.2
    ref = oracle.enuf(r, q, L, alpha, k_cut, n, m, "kaiser_bessel", 1.5, variant=variant, use_dft=True)
    Es, F = sharded_eval(enuf, torch, r, q, world,
                         lambda cnt: enuf.Plan(cnt, L, alpha, k_cut, M, sigma=1.5, m=m, dtype=torch.float64, variant=variant))
    assert all(E == Es[0] for E in Es)
    assert abs(Es[0] - ref["E"]) <= 1e-12 * abs(ref["E"])
    assert rel_rms(F, ref["F"]) <= 1e-11


def test_sharded_fp32_with_an_empty_rank(enuf, torch_cuda, oracle):
    """20k-particle fp32 Kaiser-Bessel m = 6 gas over 3 ranks, the last of which owns no particle."""
    torch = torch_cuda
    N, L = 20000, 30.0
    r, q = random_neutral_gas(N, L, seed=11, dtype=np.float32)
    alpha, kc, M, m = 0.9, 16, 32, 6
    ref = oracle.enuf(r, q, L, alpha, kc, 64, m, "kaiser_bessel")
    mk = lambda n: enuf.Plan(n, L, alpha, kc, M, m=m, dtype=torch.float32)
    plans, parts = [], []
    for lo, hi in ((0, 12000), (12000, 20000), (20000, 20000)):
        plan = mk(hi - lo)
        rt = torch.from_numpy(np.ascontiguousarray(r[lo:hi])).cuda()
        qt = torch.from_numpy(np.ascontiguousarray(q[lo:hi])).cuda()
        Ft = torch.empty((hi - lo, 3), dtype=torch.float32, device="cuda")
        plan.spectrum_partial(rt, qt, Ft)
        plans.append(plan); parts.append(Ft)
    assert float(plans[2].spectrum_tensor().abs().max()) == 0.0
    total = plans[0].spectrum_tensor() + plans[1].spectrum_tensor() + plans[2].spectrum_tensor()
    Es, Fs = [], []
    for plan, Ft in zip(plans, parts):
        plan.spectrum_tensor().copy_(total)
        E, F = plan.forces_from_spectrum(Ft)
        Es.append(E); Fs.append(F.cpu().numpy().astype(np.float64))
        plan.close()
    assert Es[0] == Es[1] == Es[2]
    assert abs(Es[0] - ref["E"]) <= 1e-6 * abs(ref["E"])
    assert rel_rms(np.concatenate(Fs, axis=0), ref["F"]) <= 2e-6


def test_sharded_call_through_a_one_rank_nccl_group(enuf, torch_cuda, oracle):
    """Plan.energy_forces_sharded with torch.distributed initialised (NCCL, world size 1): the call
    sequence of the N-GPU path, including the collective helper, equals the single-call path."""
    torch = torch_cuda
    import torch.distributed as dist
    w = make_workload("cfg1")
    rt = torch.from_numpy(w.r).cuda(); qt = torch.from_numpy(w.q).cuda()
    plan = enuf.Plan.from_workload(w)
    E0, F0 = plan.energy_forces(rt, qt)
    F0 = F0.clone()
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    started = not dist.is_initialized()
    if started:
        dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    try:
        E1, F1 = plan.energy_forces_sharded(rt, qt)
        buf = plan.spectrum_tensor()
        assert buf.is_cuda and buf.dtype == torch.float64 and buf.numel() == 2 * w.n * (2 * w.k_cut + 1) * 16
        enuf.all_reduce_sum_(buf)          # world size 1: identity
    finally:
        if started:
            dist.destroy_process_group()
    assert abs(E1 - E0) <= 1e-13 * abs(E0)
    assert rel_rms(F1.cpu().numpy(), F0.cpu().numpy()) <= 1e-12
    plan.close()


def test_finish_without_partial_is_a_state_error(enuf, torch_cuda):
    torch = torch_cuda
    w = make_workload("cfg1")
    plan = enuf.Plan.from_workload(w)
    F = torch.empty((w.N, 3), dtype=torch.float64, device="cuda")
    with pytest.raises(enuf.EnufError) as ei:
        plan.forces_from_spectrum(F)
    assert ei.value.code == enuf.ESTATE
    plan.energy_forces(torch.from_numpy(w.r).cuda(), torch.from_numpy(w.q).cuda())
    with pytest.raises(enuf.EnufError):
        plan.forces_from_spectrum(F)      # a full evaluation does not arm the second half either
    plan.close()


# ------------------------------------------------------------------ two ranks, a real collective

def _two_ranks(backend, case, tmp_path, oracle, tol_f, tol_e):
    """Spawn two ranks (tests/sharded_worker.py), each evaluating its half through Plan.energy_forces_sharded;
    both must report the same E, and the concatenated forces must match Oracle B on the whole system."""
    from sharded_worker import case_inputs
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]
    worker = os.path.join(os.path.dirname(os.path.abspath(__file__)), "sharded_worker.py")
    procs = [subprocess.Popen([sys.executable, worker, str(rk), "2", backend, str(port), case, str(tmp_path)],
                              stdout=subprocess.PIPE, stderr=subprocess.STDOUT) for rk in range(2)]
    outs = [p.communicate(timeout=600)[0].decode(errors="replace") for p in procs]
    assert all(p.returncode == 0 for p in procs), "\n".join(outs)
    r, q, pk = case_inputs(case)
    ref = oracle.enuf(r, q, pk["L"], pk["alpha"], pk["k_cut"], int(round(pk["sigma"] * pk["M"])), pk["m"], pk["window"],
                      pk["sigma"])
    parts = [np.load(os.path.join(str(tmp_path), f"rank{rk}.npz")) for rk in range(2)]
    assert float(parts[0]["E"]) == float(parts[1]["E"])                   # identical on both ranks
    assert abs(float(parts[0]["E"]) - ref["E"]) <= tol_e * abs(ref["E"])
    assert int(parts[0]["hi"]) == int(parts[1]["lo"])
    F = np.concatenate([parts[0]["F"], parts[1]["F"]], axis=0)
    assert rel_rms(F, ref["F"]) <= tol_f


@pytest.mark.parametrize("case,tol_f,tol_e", [("cfg1", 1e-11, 1e-12), ("gas20k", 2e-6, 1e-6)])
def test_two_ranks_gloo_one_gpu(torch_cuda, oracle, tmp_path, case, tol_f, tol_e):
    """Two processes on the same GPU, all-reduce of the partial spectra over gloo (CUDA tensors)."""
    _two_ranks("gloo", case, tmp_path, oracle, tol_f, tol_e)


@pytest.mark.parametrize("case,tol_f,tol_e", [("cfg1", 1e-11, 1e-12), ("gas20k", 2e-6, 1e-6)])
def test_two_ranks_nccl(torch_cuda, oracle, tmp_path, case, tol_f, tol_e):
    """Two GPUs, the all-reduce over NCCL: the path `bench.py --gpus 2` measures."""
    if torch_cuda.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    _two_ranks("nccl", case, tmp_path, oracle, tol_f, tol_e)
