"""CPU-only checks of the C-ABI library libenuf_b200.so: it loads, exports every symbol
include/enuf.h declares, validates arguments, and fails loudly (no CPU fallback) when a
compute call is made without a CUDA device.  No GPU compute here."""
import ctypes as C
import math
import os
import re

import pytest

import paper_2004_12484_b200 as enuf

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2004_12484_b200 import build
    build.build()
    return enuf.lib()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "enuf.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(enuf_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared_symbols()
    assert len(names) >= 17
    for name in names:
        assert hasattr(lib, name), name
    assert sorted(enuf.SYMBOLS) == names


def test_plan_create_validation(lib):
    h = C.c_void_p()
    bad = [
        dict(N=-1), dict(L=0.0), dict(L=float("nan")), dict(alpha=-1.0), dict(k_cut=0), dict(k_cut=9),
        dict(M=17), dict(sigma=1.0), dict(m=0), dict(m=7), dict(M=256),
    ]
    base = dict(N=10, L=10.0, alpha=0.6, k_cut=8, M=16, sigma=2.0, m=4)
    for change in bad:
        a = dict(base, **change)
        rc = lib.enuf_plan_create(C.byref(h), a["N"], a["L"], a["alpha"], a["k_cut"], a["M"], a["sigma"], a["m"])
        assert rc == enuf.EINVAL, change
        assert h.value is None
        assert lib.enuf_last_error() != b""
    rc = lib.enuf_plan_create(C.byref(h), *[base[k] for k in ("N", "L", "alpha", "k_cut", "M", "sigma", "m")])
    assert rc == enuf.OK and h.value
    assert lib.enuf_plan_set(h, 99, 0.0) == enuf.EINVAL
    assert lib.enuf_plan_set(h, enuf.OPT_WINDOW, 5.0) == enuf.EINVAL
    assert lib.enuf_plan_set(h, enuf.OPT_NUM_PARTICLES, 11.0) == enuf.EINVAL
    assert lib.enuf_plan_set(h, enuf.OPT_NUM_PARTICLES, 7.0) == enuf.OK
    assert lib.enuf_plan_set(h, enuf.OPT_SLATER_LAMBDA, -0.5) == enuf.EINVAL
    assert lib.enuf_plan_set(h, enuf.OPT_CUDA_GRAPH, 1.0) == enuf.OK   # host flag only: nothing is captured yet
    assert lib.enuf_plan_set(h, enuf.OPT_CUDA_GRAPH, 0.0) == enuf.OK
    E = C.c_double()
    assert lib.enuf_plan_energy(h, C.byref(E)) == enuf.ESTATE       # nothing evaluated yet
    assert lib.enuf_energy_forces(h, None, None, None, C.byref(E)) == enuf.EINVAL   # NULL pointers, N > 0
    lib.enuf_plan_destroy(h)
    lib.enuf_plan_destroy(None)                                     # harmless


def test_no_cpu_fallback(lib):
    """Without a CUDA device every compute call fails with ENUF_ECUDA (loudly)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    h = C.c_void_p()
    assert lib.enuf_plan_create(C.byref(h), 4, 10.0, 0.6, 8, 16, 2.0, 4) == enuf.OK
    buf = (C.c_float * 64)()
    E = C.c_double()
    rc = lib.enuf_energy_forces_host(h, buf, buf, buf, C.byref(E))
    assert rc == enuf.ECUDA
    assert b"no CPU fallback" in lib.enuf_last_error()
    lib.enuf_plan_destroy(h)
    plan = enuf.Plan(4, 10.0, 0.6, 8, 16, m=4)
    with pytest.raises((enuf.EnufError, TypeError)):
        plan.energy_forces(torch.zeros(4, 3), torch.zeros(4))


def test_parameter_rule_literals(lib):
    """Eq. 31-32 against the literal plan parameters of the configs."""
    from enuf_inputs import make_workload
    for name in ("cfg3", "cfg4"):
        w = make_workload(name)
        assert enuf.ncut(w.alpha, w.L, w.meta["delta"]) == w.k_cut
    a = enuf.alpha_from_rc(10.0, 1e-4)
    assert abs(a - 0.30348542587702925) < 1e-15
    assert enuf.ncut(a, 215.0, 1e-4) == 64
    assert abs(enuf.rc_from_ncut(64, a, 215.0) - math.pi * 64 / (a * a * 215.0)) < 1e-12
    assert enuf.ncut(-1.0, 1.0, 0.5) < 0 and math.isnan(enuf.alpha_from_rc(0.0, 0.5))


def test_plan_create_auto_reproduces_the_config_literals(lib):
    """enuf_plan_create_auto (the parameter loop of PAPER.md:350, Eq. 31-32 :254-262) against the literal plan
    parameters BASELINE.json / DESIGN.md section 2 give for configs 3, 4 and 5 (no GPU needed: plans are host objects)."""
    from enuf_inputs import make_workload
    v = C.c_double()

    def get(h, key):
        assert lib.enuf_plan_get(h, key, C.byref(v)) == enuf.OK
        return v.value

    for name in ("cfg3", "cfg4", "cfg5"):
        w = make_workload(name)
        delta = w.meta["delta"]
        r_c = math.sqrt(-math.log(delta)) / w.alpha          # Eq. 32 (R15), the cutoff the config's alpha belongs to
        h = C.c_void_p()
        assert lib.enuf_plan_create_auto(C.byref(h), w.N, w.L, delta, r_c, w.sigma, w.m) == enuf.OK
        assert abs(get(h, enuf.GET_ALPHA) - w.alpha) <= 1e-14 * w.alpha
        assert get(h, enuf.GET_K_CUT) == w.k_cut and get(h, enuf.GET_M) == w.M
        assert get(h, enuf.GET_GRID) == w.n and get(h, enuf.GET_SUPPORT) == w.m
        lib.enuf_plan_destroy(h)
    # config 5 from its own literals: r_c = 10, delta = 1e-4, L = 215
    h = C.c_void_p()
    assert lib.enuf_plan_create_auto(C.byref(h), 1000000, 215.0, 1e-4, 10.0, 2.0, 6) == enuf.OK
    assert abs(get(h, enuf.GET_ALPHA) - 0.30348542587702925) < 1e-15 and get(h, enuf.GET_K_CUT) == 64
    assert get(h, enuf.GET_M) == 128 and get(h, enuf.GET_GRID) == 256
    lib.enuf_plan_destroy(h)
    # the same rule at sigma_s = 1.5: M = 128 on the 192^3 grid (the mixed-radix FFT path)
    h = C.c_void_p()
    assert lib.enuf_plan_create_auto(C.byref(h), 1000000, 215.0, 1e-4, 10.0, 1.5, 6) == enuf.OK
    assert get(h, enuf.GET_M) == 128 and get(h, enuf.GET_GRID) == 192
    lib.enuf_plan_destroy(h)
    # ... and for an orthorhombic box
    h = C.c_void_p()
    Lb = (C.c_double * 3)(10.0, 12.0, 10.0)
    assert lib.enuf_plan_create_box(C.byref(h), 10, Lb, 1.0, 8, 32, 1.5, 4) == enuf.OK
    lib.enuf_plan_destroy(h)
    # bad arguments, and a grid the library does not have (sigma M = 512)
    h = C.c_void_p()
    assert lib.enuf_plan_create_auto(C.byref(h), 10, 215.0, 1.5, 10.0, 2.0, 6) == enuf.EINVAL
    assert lib.enuf_plan_create_auto(C.byref(h), 10, 215.0, 1e-4, 0.0, 2.0, 6) == enuf.EINVAL
    assert lib.enuf_plan_create_auto(C.byref(h), 10, 430.0, 1e-4, 10.0, 2.0, 6) == enuf.EINVAL
    assert b"sigma*M" in lib.enuf_last_error()
    assert lib.enuf_plan_get(None, enuf.GET_ALPHA, C.byref(v)) == enuf.EINVAL


def test_spread_decomposition_covers_every_slab_once():
    """The spreading kernel's pieces, checked on the host for every grid size, window, precision,
    device sizes from 1 to 200 SMs and several ENUF_OPT_SPREAD_ZCHUNK values: every (column, plane) slab in exactly one
    piece, no piece shorter than the planes it shares, every piece start zeroed; the default shares are balanced."""
    import ctypes as C
    import paper_2004_12484_b200 as enuf
    lib = enuf.lib()
    G, lo, hi = C.c_int(), C.c_int(), C.c_int()
    for n in (32, 48, 64, 96, 128, 192, 256, 384):
        for m in (1, 2, 4, 6):
            for prec in (enuf.F32, enuf.F64):
                trim = 1 if (prec == enuf.F32 and m >= 5) else 0
                for sms in (1, 7, 20, 108, 132, 148, 200):
                    rc = lib.enuf_spread_split_check(n, m, prec, trim, sms, 0, C.byref(G), C.byref(lo), C.byref(hi))
                    assert rc == enuf.OK, (n, m, prec, sms, lib.enuf_last_error())
                    ncol = (n // (32 if n >= 128 else 16)) * (n // 16)
                    assert 1 <= G.value <= max(ncol * n // (2 * m - trim + 1), 1)
                    # balanced: the most loaded CTA is within a piece's minimum length (or 15 %) of the least loaded one
                    assert hi.value - lo.value <= max(2 * m, 0.15 * hi.value) or G.value <= ncol, (n, m, sms, G.value, lo.value, hi.value)
                for z in (1, 5, 16, n):
                    rc = lib.enuf_spread_split_check(n, m, prec, trim, 148, z, C.byref(G), None, None)
                    assert rc == enuf.OK, (n, m, prec, z, lib.enuf_last_error())
    # the headline configuration: 288 CTAs of 112 .. 114 slabs on a 148-SM device
    assert lib.enuf_spread_split_check(256, 6, enuf.F32, 1, 148, 0, C.byref(G), C.byref(lo), C.byref(hi)) == enuf.OK
    assert (G.value, lo.value, hi.value) == (288, 112, 114)
    assert lib.enuf_spread_split_check(40, 6, enuf.F32, 1, 148, 0, None, None, None) == enuf.EINVAL
