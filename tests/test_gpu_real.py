"""GPU parity of the real-space Ewald part (enuf_real_space) against Oracle R
(oracle.real_forces / real_energy / self_energy), and the full Ewald sum on the device:
E_real + E_rec - E_self of rock salt reproduces the Madelung constant (Eq. 25).

Bars: fp64 relative RMS force error <= 1e-12, energies 1e-13; fp32 <= 2e-6 / 1e-6 (the path's fp32 bar).
"""
import math

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


def gpu_real(enuf, torch, r, q, L, alpha, r_cut, dtype, lam=0.0, **kw):
    plan = enuf.Plan(q.shape[0], L, alpha, 4, 16, m=4, dtype=dtype, slater_lambda=lam)
    Er, Es, F = plan.real_space(torch.from_numpy(r).cuda(), torch.from_numpy(q).cuda(), r_cut, **kw)
    out = (Er, Es, F.cpu().numpy().astype(np.float64))
    plan.close()
    return out


@pytest.mark.parametrize("N,L,r_cut,lam", [(300, 6.0, 3.0, 0.0),      # r_cut = L/2: one cell, all pairs
                                            (2000, 12.0, 2.2, 0.0),    # 10 cells per dimension, s = 2
                                            (2000, 12.0, 2.4, 0.25),   # exactly 10 cells; Slater factors
                                            (1500, 11.0, 4.3, 0.0)])   # 5 cells: every cell is a neighbour
def test_real_space_fp64_matches_oracle(enuf, torch_cuda, oracle, N, L, r_cut, lam):
    torch = torch_cuda
    alpha = 2.6 / r_cut
    r, q = random_neutral_gas(N, L, seed=N + 1)
    e_i, F_ref = oracle.real_forces(r, q, L, alpha, r_cut, shells=1, slater_lambda=lam)
    Er, Es, F = gpu_real(enuf, torch, r, q, L, alpha, r_cut, torch.float64, lam)
    assert rel_rms(F, F_ref) <= 1e-12
    assert abs(Er - e_i.sum()) <= 1e-13 * np.abs(e_i).sum()
    assert abs(Es - oracle.self_energy(q, alpha)) <= 1e-14 * Es
    if lam == 0.0:
        assert abs(Er - oracle.real_energy(r, q, L, alpha, r_cut, 1)) <= 1e-12 * np.abs(e_i).sum()
    assert np.abs(F.sum(axis=0)).max() <= 1e-11 * np.abs(F).max()        # Newton's third law


def test_real_space_fp32_matches_oracle(enuf, torch_cuda, oracle):
    """8000 charges at density 0.1 (config 5's), r_cut = 10, alpha from delta = 1e-4: every particle."""
    torch = torch_cuda
    N, L, r_cut = 8000, 43.0, 10.0
    alpha = math.sqrt(-math.log(1e-4)) / r_cut
    r, q = random_neutral_gas(N, L, seed=21, dtype=np.float32)
    e_i, F_ref = oracle.real_forces(r, q, L, alpha, r_cut, shells=1)
    Er, Es, F = gpu_real(enuf, torch, r, q, L, alpha, r_cut, torch.float32)
    assert rel_rms(F, F_ref) <= 2e-6
    assert abs(Er - e_i.sum()) <= 1e-6 * np.abs(e_i).sum()
    assert abs(Es - oracle.self_energy(q, alpha)) <= 1e-12 * Es


def test_real_space_fp32_large_sampled(enuf, torch_cuda, oracle):
    """100 000 charges in L = 100 (density 0.1): 20 cells per dimension; 256 sampled particles."""
    torch = torch_cuda
    N, L, r_cut = 100_000, 100.0, 10.0
    alpha = math.sqrt(-math.log(1e-4)) / r_cut
    r, q = random_neutral_gas(N, L, seed=22, dtype=np.float32)
    sample = np.random.default_rng(5).choice(N, 256, replace=False)
    _, F_ref = oracle.real_forces(r, q, L, alpha, r_cut, shells=1, sample=sample)
    _, _, F = gpu_real(enuf, torch, r, q, L, alpha, r_cut, torch.float32)
    assert rel_rms(F[sample], F_ref) <= 2e-6


def test_madelung_constant_on_the_device(enuf, torch_cuda):
    """Eq. 25 on the GPU in fp64: rock salt, 8^3 cells (R18, R20):
    -(E_real + E_rec - E_self) r0 / (N/2) = 1.747565 to 1e-6 (BASELINE north_star)."""
    torch = torch_cuda
    w = make_workload("cfg2_perfect_k16")
    plan = enuf.Plan.from_workload(w)
    r = torch.from_numpy(w.r).cuda(); q = torch.from_numpy(w.q).cuda()
    E_rec, F = plan.energy_forces(r, q)
    E_real, E_self, F = plan.real_space(r, q, w.L / 2, F=F, accumulate=True)
    madelung = -(E_real + E_rec - E_self) * w.meta["r0"] / (w.N / 2)
    assert abs(madelung - 1.7475645946331822) < 1e-6
    assert float(F.abs().max()) < 1e-9          # perfect lattice: every total force vanishes by symmetry
    plan.close()


def test_real_space_accumulate_neutral_wrap_and_errors(enuf, torch_cuda, oracle):
    torch = torch_cuda
    N, L, r_cut, alpha = 1200, 12.0, 2.4, 1.1
    r, q = random_neutral_gas(N, L, seed=8)
    q[::5] = 0.0                                                 # neutral particles: no force, exert none
    shift = np.random.default_rng(1).integers(-2, 3, size=r.shape) * L
    _, F_ref = oracle.real_forces(r, q, L, alpha, r_cut, shells=1)
    plan = enuf.Plan(N, L, alpha, 4, 16, m=4, dtype=torch.float64)
    rt = torch.from_numpy(r + shift).cuda(); qt = torch.from_numpy(q).cuda()    # images of the same system
    _, _, F = plan.real_space(rt, qt, r_cut)
    assert rel_rms(F.cpu().numpy(), F_ref) <= 1e-11
    assert float(F[::5].abs().max()) == 0.0
    F0 = torch.full((N, 3), 2.0, dtype=torch.float64, device="cuda")
    plan.real_space(rt, qt, r_cut, F=F0, accumulate=True, want_energy=False)
    assert rel_rms((F0 - 2.0).cpu().numpy(), F_ref) <= 1e-11
    with pytest.raises(enuf.EnufError) as ei:
        plan.real_space(rt, qt, 0.51 * L)
    assert ei.value.code == enuf.EINVAL
    plan.set_num_particles(0)
    Er, Es, _ = plan.real_space(rt[:0].contiguous(), qt[:0].contiguous(), r_cut)
    assert Er == 0.0 and Es == 0.0
    plan.close()
