"""enuf_self_energy_static: the allocation-free entry point (static device scratch) against the existing path,
enuf_real_space's E_self.  Collected last on purpose (the suite runs with pytest -x): a failure here hides nothing."""
import ctypes as C
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

E_TOL = 1e-12          # the fp64 energy tolerance of the parity tests (F64_E, tests/test_gpu_parity.py)


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def enuf(torch_cuda):
    import paper_2004_12484_b200 as e
    e.lib()   # fails loudly if the library has not been built
    return e


def _existing_path(enuf, torch, q, alpha):
    """E_self as enuf_real_space returns it (plan workspace from cudaMalloc)."""
    N, L = q.shape[0], 9.0
    g = torch.Generator(device="cpu").manual_seed(N)
    r = (torch.rand((N, 3), generator=g, dtype=torch.float64) * L).to(q.dtype).cuda()
    plan = enuf.Plan(N, L, alpha, 8, 16, sigma=2.0, m=2, dtype=q.dtype)
    _, E_self, _ = plan.real_space(r, q, 0.5)
    plan.close()
    return E_self


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_two_calls_in_a_row_match_the_existing_path(enuf, torch_cuda, dtype):
    torch = torch_cuda
    tdt = torch.float32 if dtype == "f32" else torch.float64
    rng = np.random.default_rng(20)
    alpha = 0.85
    out = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    # the second call is shorter than the first: the scratch still holds the first call's partial sums
    for N in (300007, 4099):
        q = torch.from_numpy(rng.uniform(-1.5, 1.5, size=N)).to(tdt).cuda()
        q[::7] = 0
        enuf.self_energy_static(q, alpha, out)
        got = out.item()
        want = _existing_path(enuf, torch, q, alpha)
        assert abs(got - want) <= E_TOL * abs(want)
        # and the definition itself, Eq. 24, summed in fp64 by numpy
        ref = alpha / math.sqrt(math.pi) * float((q.cpu().double().numpy() ** 2).sum())
        assert abs(got - ref) <= E_TOL * abs(ref)
    # same input again: the fixed summation order makes the result reproducible bit by bit
    enuf.self_energy_static(q, alpha, out)
    assert out.item() == got


def test_empty_input_and_limits(enuf, torch_cuda):
    torch = torch_cuda
    out = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    enuf.self_energy_static(torch.empty(0, dtype=torch.float32, device="cuda"), 1.0, out)
    assert out.item() == 0.0
    lib = enuf.lib()
    q = torch.ones(8, dtype=torch.float32, device="cuda")
    too_many = enuf.SELF_STATIC_MAX_N + 1      # refused before anything is launched or read
    rc = lib.enuf_self_energy_static(C.c_void_p(q.data_ptr()), too_many, enuf.F32, 1.0, None, C.c_void_p(out.data_ptr()))
    assert rc == enuf.EINVAL and b"ENUF_SELF_STATIC_MAX_N" in lib.enuf_last_error()
    assert lib.enuf_self_energy_static(C.c_void_p(q.data_ptr()), 8, enuf.F32, 1.0, None, None) == enuf.EINVAL
    assert lib.enuf_self_energy_static(None, 8, enuf.F32, 1.0, None, C.c_void_p(out.data_ptr())) == enuf.EINVAL
    assert lib.enuf_self_energy_static(C.c_void_p(q.data_ptr()), 8, 7, 1.0, None, C.c_void_p(out.data_ptr())) == enuf.EINVAL
    torch.cuda.synchronize()
    assert out.item() == 0.0                   # the refused calls wrote nothing
    # the largest N the array was built for runs (16384 CTAs)
    big = torch.full((enuf.SELF_STATIC_MAX_N,), 0.5, dtype=torch.float32, device="cuda")
    enuf.self_energy_static(big, 2.0, out)
    ref = 2.0 / math.sqrt(math.pi) * 0.25 * enuf.SELF_STATIC_MAX_N
    assert abs(out.item() - ref) <= E_TOL * ref
