"""Pins for the CPU oracle (oracle/enuf_oracle.c) against things other than itself:
closed forms, values fixed by the paper / task statement (tests/golden/paper_values.txt),
invariants, finite differences, quadrature, numpy.fft and brute force.  CPU only.
"""
import math
import os

import numpy as np
import pytest
from scipy import integrate

from enuf_inputs import make_workload, random_neutral_gas

GOLDEN = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")) as fh:
    for line in fh:
        line = line.split("#")[0].strip()
        if "=" in line:
            k, v = line.split("=")
            GOLDEN[k.strip()] = float(v)


# ----------------------------------------------------------------- Oracle A: energy

def _total_ewald(O, r, q, L, alpha, k_cut, r_cut, shells):
    e_rec, _ = O.direct(r, q, L, alpha, k_cut, forces=False)
    return O.real_energy(r, q, L, alpha, r_cut, shells) + e_rec - O.self_energy(q, alpha)


@pytest.mark.parametrize("name,tol", [("cfg2_perfect", 1e-6), ("cfg2_perfect_k16", 1e-9)])
def test_madelung_rock_salt(oracle, name, tol):
    """Full Ewald energy (real + reciprocal - self, Eq. 25) of rock salt
    reproduces the Madelung constant (BASELINE north_star: 1.747565 to 1e-6)."""
    w = make_workload(name)
    e = _total_ewald(oracle, w.r, w.q, w.L, w.alpha, w.k_cut, r_cut=w.L / 2, shells=1)
    madelung = -e * w.meta["r0"] / (w.N / 2)
    assert abs(madelung - GOLDEN["madelung_nacl"]) < 1e-6
    assert abs(madelung - 1.7475645946331822) < tol   # more digits of the same constant


@pytest.mark.parametrize("alpha", [2.0, 3.0, 5.0])
def test_wigner_single_charge(oracle, alpha):
    """One charge in a unit cube with neutralising background: E = -xi/(2L)."""
    L = 1.0
    r = np.array([[0.3, 0.55, 0.8]]); q = np.array([1.0])
    k_cut = 14
    e_rec, _ = oracle.direct(r, q, L, alpha, k_cut, forces=False)
    e = (e_rec + oracle.real_energy(r, q, L, alpha, 6.0, 6) - oracle.self_energy(q, alpha)
         - math.pi / (2 * alpha ** 2 * L ** 3))
    assert abs(e + GOLDEN["wigner_cubic"] / (2 * L)) < 2e-9


def test_total_energy_independent_of_alpha(oracle):
    """PAPER.md:467 'the electrostatic energy is invariant to alpha'."""
    r, q = random_neutral_gas(24, 3.0, seed=77)
    L = 3.0
    es = [_total_ewald(oracle, r, q, L, a, k_cut=kc, r_cut=3 * L, shells=3)
          for a, kc in ((1.4, 10), (2.0, 14), (2.6, 18))]
    assert max(es) - min(es) < 1e-9 * abs(es[0])


def test_parameter_rule(oracle):
    """Eq. 31-32: literals of the configs and the paper's alpha >= 0.12."""
    for name in ("cfg3", "cfg4", "cfg5"):
        w = make_workload(name) if name != "cfg5" else None
        if name == "cfg5":
            a = oracle.alpha_from_rc(10.0, 1e-4)
            assert abs(a - 0.30348542587702925) < 1e-15
            assert oracle.ncut(a, 215.0, 1e-4) == 64
        else:
            assert oracle.ncut(w.alpha, w.L, w.meta["delta"]) == w.k_cut
    r_c = GOLDEN["dpd_rc_over_Rc"] * GOLDEN["dpd_beta"] * GOLDEN["dpd_lambda_e"]
    a = oracle.alpha_from_rc(r_c, GOLDEN["dpd_delta"])
    assert GOLDEN["dpd_alpha_min"] <= a < GOLDEN["dpd_alpha_min"] + 0.01   # prints "0.12"


# ----------------------------------------------------------------- Oracle A: forces

def test_direct_forces_are_minus_gradient(oracle):
    r, q = random_neutral_gas(12, 4.0, seed=5)
    L, alpha, kc = 4.0, 1.1, 6
    _, F = oracle.direct(r, q, L, alpha, kc)
    h = 1e-5
    for i in (0, 5, 11):
        for d in range(3):
            rp = r.copy(); rp[i, d] += h
            rm = r.copy(); rm[i, d] -= h
            ep, _ = oracle.direct(rp, q, L, alpha, kc, forces=False)
            em, _ = oracle.direct(rm, q, L, alpha, kc, forces=False)
            assert abs(F[i, d] + (ep - em) / (2 * h)) < 2e-9 * np.abs(F).max()


def test_direct_momentum_and_antisymmetry(oracle):
    r, q = random_neutral_gas(64, 5.0, seed=9)
    _, F = oracle.direct(r, q, 5.0, 1.0, 7)
    assert np.abs(F.sum(0)).max() < 1e-10 * np.abs(F).max()          # 'momentum conserved' :79
    r2 = np.array([[0.1, 0.2, 0.3], [1.7, 2.9, 0.4]]); q2 = np.array([1.0, -1.0])
    _, F2 = oracle.direct(r2, q2, 5.0, 1.0, 7)
    assert np.abs(F2[0] + F2[1]).max() < 1e-13 * np.abs(F2).max()


def test_direct_sampled_forces_match_full(oracle):
    r, q = random_neutral_gas(32, 5.0, seed=10)
    _, F = oracle.direct(r, q, 5.0, 1.0, 6)
    _, Fs = oracle.direct(r, q, 5.0, 1.0, 6, sample=[3, 30, 7])
    assert np.array_equal(Fs, F[[3, 30, 7]])


def test_direct_S_single_particle_closed_form(oracle):
    """S(n) of one charge is exp(-2 pi i n.x) (Eq. 37)."""
    r = np.array([[1.0, 2.5, 7.0]]); q = np.array([2.0]); L = 10.0
    S = oracle.direct_S(r, q, L, [[1, 0, 0], [0, 1, 0], [0, 0, 1], [1, -2, 3]])
    x = r[0] / L
    exp = [2 * np.exp(-2j * np.pi * np.dot(n, x)) for n in ([1, 0, 0], [0, 1, 0], [0, 0, 1], [1, -2, 3])]
    assert np.allclose(S, exp, rtol=0, atol=1e-14)


# ----------------------------------------------------------------- windows

@pytest.mark.parametrize("window,m,tol", [("kaiser_bessel", 4, 1e-8), ("kaiser_bessel", 6, 1e-11),
                                          ("kaiser_bessel", 2, 1e-4), ("gaussian", 4, 1e-11),
                                          ("gaussian", 6, 1e-11)])
def test_window_transform_by_quadrature(oracle, window, m, tol):
    """Phi(k) is the continuous Fourier transform of phi (R6), checked by quadrature."""
    n, sigma = 64, 2.0
    lim = m if window == "kaiser_bessel" else 30.0
    for k in (0, 1, 5, 16):
        f = lambda d: oracle.phi(window, m, sigma, d) * math.cos(2 * math.pi * k * d / n)
        val, _ = integrate.quad(f, -lim, lim, limit=400, epsabs=1e-13, epsrel=1e-13)
        ref = oracle.Phi(window, m, sigma, n, k)
        assert abs(val - ref) < tol * abs(oracle.Phi(window, m, sigma, n, 0)), (k, val, ref)


# ----------------------------------------------------------------- B-spline window

def test_bspline_m1_is_the_hat_function(oracle):
    """Order 2 (m = 1): phi(d) = 1 - |d| on [-1, 1] -- a closed form the recursion must reproduce."""
    for d in (-1.3, -1.0, -0.75, -0.2, 0.0, 0.4, 0.999, 1.0, 2.0):
        want = max(0.0, 1.0 - abs(d))
        assert abs(oracle.phi("bspline", 1, 2.0, d) - want) < 1e-15
    assert oracle.dphi("bspline", 1, 2.0, 0.3) == -1.0 and oracle.dphi("bspline", 1, 2.0, -0.3) == 1.0


@pytest.mark.parametrize("m", [2, 3, 4, 6])
def test_bspline_partition_of_unity_and_support(oracle, m):
    """sum_j B_p(x - j) = 1 for every x (the classic B-spline identity), phi(0) = 1 (R7), support [-m, m],
    central value of the cubic spline 2/3 (phi = B_4 / B_4(0), so phi(1) = (1/6)/(2/3) = 1/4)."""
    B0 = 1.0 / sum(oracle.phi("bspline", m, 2.0, j) for j in range(-m, m + 1))     # = B_2m(0)
    for x in (0.0, 0.17, 0.5, 0.93):
        total = sum(oracle.phi("bspline", m, 2.0, x - j) for j in range(-m - 1, m + 2)) * B0
        assert abs(total - 1.0) < 1e-14
    assert abs(oracle.phi("bspline", m, 2.0, 0.0) - 1.0) < 1e-15
    assert oracle.phi("bspline", m, 2.0, m) == 0.0 and oracle.phi("bspline", m, 2.0, m + 0.3) == 0.0
    assert oracle.phi("bspline", m, 2.0, m - 1e-3) > 0.0
    if m == 2:
        assert abs(B0 - 2.0 / 3.0) < 1e-15 and abs(oracle.phi("bspline", 2, 2.0, 1.0) - 0.25) < 1e-15


@pytest.mark.parametrize("m", [2, 4, 6])
def test_bspline_transform_and_derivative(oracle, m):
    n = 64
    for k in (0, 1, 5, 16):
        f = lambda d: oracle.phi("bspline", m, 2.0, d) * math.cos(2 * math.pi * k * d / n)
        val, _ = integrate.quad(f, -m, m, limit=400, epsabs=1e-13, epsrel=1e-13, points=list(range(-m + 1, m)))
        assert abs(val - oracle.Phi("bspline", m, 2.0, n, k)) < 1e-11 * oracle.Phi("bspline", m, 2.0, n, 0)
    h = 1e-6
    for d in (-m + 0.4, -0.7, 0.0, 0.3, 1.5, m - 0.2):
        fd = (oracle.phi("bspline", m, 2.0, d + h) - oracle.phi("bspline", m, 2.0, d - h)) / (2 * h)
        assert abs(fd - oracle.dphi("bspline", m, 2.0, d)) < 1e-8


@pytest.mark.parametrize("variant,bound", [("analytic", 2e-2), ("ik", 2e-3)])
def test_bspline_enuf_against_direct_ewald(oracle, variant, bound):
    """Brute force: Oracle B with the B-spline window (m = 6, sigma = 2) against Oracle A on 64 particles.
    The B-spline is the least accurate of the NFFT windows at equal m (error ~ (1/(2 sigma - 1))^{2m} ~ 2e-6 per
    dimension at the band edge)."""
    L, alpha, kc, n, m = 6.0, 1.0, 8, 32, 6
    r, q = random_neutral_gas(64, L, seed=21)
    Ea, Fa = oracle.direct(r, q, L, alpha, kc)
    b = oracle.enuf(r, q, L, alpha, kc, n, m, "bspline", variant=variant)
    assert abs(b["E"] - Ea) < 1e-3 * abs(Ea)
    err = math.sqrt(((b["F"] - Fa) ** 2).sum() / (Fa ** 2).sum())
    assert err < bound, err
    if variant == "analytic":       # exact gradient of the ENUF energy (R17)
        h = 1e-5
        for i, d in ((3, 0), (40, 2)):
            rp = r.copy(); rp[i, d] += h
            rm = r.copy(); rm[i, d] -= h
            ep = oracle.enuf(rp, q, L, alpha, kc, n, m, "bspline", forces=False)["E"]
            em = oracle.enuf(rm, q, L, alpha, kc, n, m, "bspline", forces=False)["E"]
            assert abs(b["F"][i, d] + (ep - em) / (2 * h)) < 1e-7 * np.abs(b["F"]).max()


# ----------------------------------------------------------------- oversampling 1.5: grids that are not powers of two

@pytest.mark.parametrize("n", [12, 24, 48])
def test_dft_line_any_length_equals_numpy(oracle, n):
    """The oracle's plain DFT line transform (the definition, Eq. 34-35 convention R11) for lengths 3 * 2^k, the grids
    of sigma_s = 1.5, against numpy.fft in both directions; and a 3-D transform with the axis order."""
    rng = np.random.default_rng(n)
    x = rng.normal(size=n) + 1j * rng.normal(size=n)
    assert np.abs(oracle.fft_line(x, -1, True) - np.fft.fft(x)).max() < 1e-12
    assert np.abs(oracle.fft_line(x, +1, True) - np.fft.ifft(x) * n).max() < 1e-12
    if n <= 24:
        a = rng.normal(size=(n, n, n)) + 1j * rng.normal(size=(n, n, n))
        assert np.abs(oracle.fft3d(a, -1, True) - np.fft.fftn(a)).max() < 1e-10


@pytest.mark.parametrize("window", ["kaiser_bessel", "gaussian"])
def test_enuf_oversampling_one_and_a_half_against_direct_ewald(oracle, window):
    """sigma_s = 1.5 (M = 16, n = 24; the paper sweeps 1.5 and 2, Fig. 1): Oracle B with the DFT on the 24^3 grid against
    Oracle A.  The error falls with m and is larger than at sigma_s = 2 with the same m; the analytic forces are the
    exact gradient of the ENUF energy at any sigma (R17)."""
    L, alpha, kc, M = 6.0, 1.0, 8, 16
    r, q = random_neutral_gas(64, L, seed=21)
    Ea, Fa = oracle.direct(r, q, L, alpha, kc)
    err = {}
    for sigma in (1.5, 2.0):
        for m in (2, 4):
            b = oracle.enuf(r, q, L, alpha, kc, int(sigma * M), m, window, sigma, variant="ik", use_dft=True)
            err[sigma, m] = math.sqrt(((b["F"] - Fa) ** 2).sum() / (Fa ** 2).sum())
            assert abs(b["E"] - Ea) < (3e-3 if m == 2 else 5e-5) * abs(Ea)
    assert err[1.5, 4] < 0.05 * err[1.5, 2] and err[2.0, 4] < 0.05 * err[2.0, 2], err
    assert err[1.5, 4] > 2 * err[2.0, 4], err
    n, m, h = 24, 4, 1e-5
    b = oracle.enuf(r, q, L, alpha, kc, n, m, window, 1.5, variant="analytic", use_dft=True)
    for i, d in ((7, 2), (50, 0)):
        rp = r.copy(); rp[i, d] += h
        rm = r.copy(); rm[i, d] -= h
        ep = oracle.enuf(rp, q, L, alpha, kc, n, m, window, 1.5, forces=False, use_dft=True)["E"]
        em = oracle.enuf(rm, q, L, alpha, kc, n, m, window, 1.5, forces=False, use_dft=True)["E"]
        assert abs(b["F"][i, d] + (ep - em) / (2 * h)) < 1e-7 * np.abs(b["F"]).max()


# ----------------------------------------------------------------- sinc-power window

def test_sinc_power_m1_transform_is_the_hat_function(oracle):
    """m = 1: phi = sinc^2(pi c d), c = (2 - 1/sigma)/2.  Its transform is the textbook triangle of half-width c and
    height 1/c (int sinc^2(pi c d) dd = 1/c); at the grid frequency k/n: (1/c) max(0, 1 - |k|/(n c))."""
    for sigma, n in ((2.0, 64), (1.5, 48)):
        c = (2.0 - 1.0 / sigma) / 2.0
        for k in (0, 1, 7, 20, int(n * c), int(n * c) + 3):
            want = max(0.0, 1.0 - k / (n * c)) / c
            assert abs(oracle.Phi("sinc_power", 1, sigma, n, k) - want) < 1e-14
    # the window itself at a few points, written out
    for d in (0.25, 1.0, 1.5):
        t = math.pi * 0.75 * d
        assert abs(oracle.phi("sinc_power", 1, 2.0, d) - (math.sin(t) / t) ** 2) < 1e-15
    assert oracle.phi("sinc_power", 1, 2.0, 4.0 / 3.0) < 1e-30           # first zero of sinc(pi c d): d = 1/c


@pytest.mark.parametrize("m", [2, 3, 4, 6])
def test_sinc_power_transform_by_quadrature(oracle, m):
    """Phi(k) = int phi(d) cos(2 pi k d/n) dd over the real line (the window is not compactly supported: the integral
    is taken over |d| <= D and the tail bounded by 2 int_D^inf (pi c d)^(-2m) dd)."""
    n, sigma, D = 64, 2.0, 300.0
    c = (2.0 - 1.0 / sigma) / (2.0 * m)
    tail = 2.0 * (math.pi * c) ** (-2 * m) * D ** (1 - 2 * m) / (2 * m - 1)
    assert tail < 2e-8
    for k in (0, 1, 5, 16, 30):
        f = lambda d: oracle.phi("sinc_power", m, sigma, d) * math.cos(2 * math.pi * k * d / n)
        val, _ = integrate.quad(f, -D, D, limit=20000, epsabs=1e-13, epsrel=1e-13)
        assert abs(val - oracle.Phi("sinc_power", m, sigma, n, k)) < tail + 1e-11, (k, val)
    assert abs(oracle.phi("sinc_power", m, sigma, 0.0) - 1.0) < 1e-15     # R7


@pytest.mark.parametrize("m", [1, 2, 4, 6])
def test_sinc_power_derivative_by_differences(oracle, m):
    """phi' against central differences of phi on both branches of its evaluation (series for |pi c d| < 1/2, closed form
    beyond), continuity at the switch, oddness."""
    c = (2.0 - 0.5) / (2.0 * m)
    h = 1e-5
    for d in (-m - 0.4, -1.7, -0.3, -1e-3, 0.0, 1e-4, 0.05, 0.37, 1.0, 2.6, m - 0.5, m + 0.45):
        fd = (oracle.phi("sinc_power", m, 2.0, d + h) - oracle.phi("sinc_power", m, 2.0, d - h)) / (2 * h)
        an = oracle.dphi("sinc_power", m, 2.0, d)
        assert abs(fd - an) < 2e-9, (d, fd, an)
        assert oracle.dphi("sinc_power", m, 2.0, -d) == -an
    ds = 0.5 / (math.pi * c)                                              # the switch between the branches
    a, b = oracle.dphi("sinc_power", m, 2.0, ds * (1 - 1e-9)), oracle.dphi("sinc_power", m, 2.0, ds * (1 + 1e-9))
    assert abs(a - b) < 1e-8 * abs(a)


@pytest.mark.parametrize("variant", ["analytic", "ik"])
def test_sinc_power_enuf_against_direct_ewald(oracle, variant):
    """Brute force: Oracle B with the sinc-power window against Oracle A on 64 particles; the error falls with m
    (the stencil cuts the window at sinc(3 pi/4 (1 + 1/2m))^(2m), 3e-7 of the peak at m = 6)."""
    L, alpha, kc, n = 6.0, 1.0, 8, 32
    r, q = random_neutral_gas(64, L, seed=22)
    Ea, Fa = oracle.direct(r, q, L, alpha, kc)
    errs = []
    for m in (2, 4, 6):
        b = oracle.enuf(r, q, L, alpha, kc, n, m, "sinc_power", variant=variant)
        errs.append(math.sqrt(((b["F"] - Fa) ** 2).sum() / (Fa ** 2).sum()))
        if m == 6:
            assert abs(b["E"] - Ea) < 1e-4 * abs(Ea)
    assert errs[0] > 3 * errs[1] > 9 * errs[2], errs
    assert errs[2] < (2e-3 if variant == "analytic" else 2e-4), errs
    if variant == "analytic":       # exact gradient of the ENUF energy (R17)
        h, m = 1e-5, 4
        b = oracle.enuf(r, q, L, alpha, kc, n, m, "sinc_power", variant=variant)
        for i, d in ((5, 1), (33, 0)):
            rp = r.copy(); rp[i, d] += h
            rm = r.copy(); rm[i, d] -= h
            ep = oracle.enuf(rp, q, L, alpha, kc, n, m, "sinc_power", forces=False)["E"]
            em = oracle.enuf(rm, q, L, alpha, kc, n, m, "sinc_power", forces=False)["E"]
            assert abs(b["F"][i, d] + (ep - em) / (2 * h)) < 1e-7 * np.abs(b["F"]).max()


@pytest.mark.parametrize("window,m", [("kaiser_bessel", 4), ("kaiser_bessel", 6), ("gaussian", 4)])
def test_window_normalisation_symmetry_support(oracle, window, m):
    assert abs(oracle.phi(window, m, 2.0, 0.0) - 1.0) < 1e-15           # R7
    for d in (0.3, 1.7, m - 0.01):
        assert oracle.phi(window, m, 2.0, d) == oracle.phi(window, m, 2.0, -d)
        assert oracle.dphi(window, m, 2.0, d) == -oracle.dphi(window, m, 2.0, -d)
    if window == "kaiser_bessel":
        assert oracle.phi(window, m, 2.0, m + 0.25) == 0.0             # support radius m (R8)
        assert oracle.dphi(window, m, 2.0, m + 0.25) == 0.0


@pytest.mark.parametrize("window,m", [("kaiser_bessel", 4), ("kaiser_bessel", 6), ("gaussian", 4),
                                      ("gaussian", 6)])
def test_window_derivative_by_differences(oracle, window, m):
    h = 1e-5
    pts = [-m + 0.3, -2.2, -0.4, 0.0, 0.37, 1.0, m - 0.6, m - 1e-3, m - 1e-6]
    for d in pts:
        if window == "kaiser_bessel" and abs(d) + h >= m:
            hh = (m - abs(d)) / 4
        else:
            hh = h
        fd = (oracle.phi(window, m, 2.0, d + hh) - oracle.phi(window, m, 2.0, d - hh)) / (2 * hh)
        an = oracle.dphi(window, m, 2.0, d)
        assert abs(fd - an) < 1e-8 * max(1.0, abs(an)) + 1e-3 * abs(an) * (hh < h), (d, fd, an)


def test_kb_derivative_series_branch_is_continuous(oracle):
    """The small-s series of phi' must join the closed form (x = b s = 0.25 switch)."""
    m, b = 6, math.pi * 1.5
    s = 0.25 / b
    for eps in (1e-9, 1e-7):
        d_lo = math.sqrt(m * m - (s * (1 - eps)) ** 2)
        d_hi = math.sqrt(m * m - (s * (1 + eps)) ** 2)
        a, c = oracle.dphi("kaiser_bessel", m, 2.0, d_lo), oracle.dphi("kaiser_bessel", m, 2.0, d_hi)
        assert abs(a - c) < 1e-6 * abs(a)


def test_slater_form_factor_by_radial_quadrature(oracle):
    """R19: f(k) is the Fourier transform of Eq. 51, whose integral is q."""
    lam, L = 0.25, 20.0
    rho = lambda r: math.exp(-2 * r / lam) / (math.pi * lam ** 3)
    total, _ = integrate.quad(lambda r: 4 * math.pi * r * r * rho(r), 0, 40 * lam)
    assert abs(total - 1.0) < 1e-10
    for n2 in (1, 9, 100, 324):
        k = 2 * math.pi * math.sqrt(n2) / L
        f, _ = integrate.quad(lambda r: 4 * math.pi * r * r * rho(r) * math.sin(k * r) / (k * r),
                              1e-300, 40 * lam, epsabs=1e-14)
        assert abs(f * f - oracle.slater_f2(n2, lam, L)) < 1e-10
    assert oracle.slater_f2(50, 0.0, L) == 1.0
    assert abs(oracle.slater_f2(50, 1e-9, L) - 1.0) < 1e-12


# ----------------------------------------------------------------- Oracle B: FFT

@pytest.mark.parametrize("n", [8, 32, 64])
def test_dft_fft_numpy_agree_on_lines(oracle, n):
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    for sign, ref in ((-1, np.fft.fft(x)), (+1, np.fft.ifft(x) * n)):
        a = oracle.fft_line(x, sign, use_dft=True)
        b = oracle.fft_line(x, sign, use_dft=False)
        scale = np.abs(ref).max()
        assert np.abs(a - ref).max() < 1e-13 * scale
        assert np.abs(b - ref).max() < 1e-13 * scale


def test_fft_line_256_vs_numpy(oracle):
    rng = np.random.default_rng(256)
    x = rng.standard_normal(256) + 1j * rng.standard_normal(256)
    assert np.abs(oracle.fft_line(x, -1, False) - np.fft.fft(x)).max() < 1e-12 * np.abs(x).sum()


def test_fft3d_vs_numpy_and_axis_order(oracle):
    rng = np.random.default_rng(3)
    n = 16
    a = rng.standard_normal((n, n, n)) + 1j * rng.standard_normal((n, n, n))
    ref = np.fft.fftn(a)
    for use_dft in (True, False):
        assert np.abs(oracle.fft3d(a, -1, use_dft) - ref).max() < 1e-12 * np.abs(ref).max()
    assert np.abs(oracle.fft3d(a, +1) - np.fft.ifftn(a) * n ** 3).max() < 1e-12 * np.abs(ref).max()


# ----------------------------------------------------------------- Oracle B: spreading / S~

def test_spread_additivity_eq61(oracle):
    """Eq. 61: S (hence the spread grid) is additive over subsets."""
    w = make_workload("cfg1")
    half = w.N // 2
    g = oracle.spread(w.r, w.q, w.L, w.n, w.m, w.window)
    ga = oracle.spread(w.r[:half], w.q[:half], w.L, w.n, w.m, w.window)
    gb = oracle.spread(w.r[half:], w.q[half:], w.L, w.n, w.m, w.window)
    assert np.abs(g - (ga + gb)).max() < 1e-13 * np.abs(g).max()


def test_spread_total_mass_and_periodic_wrap(oracle):
    """sum_l g[l] = q * (sum_k phi)^3 for one particle, also when the stencil wraps."""
    for pos in ([5.2, 5.7, 5.1], [0.05, 9.99, 0.4]):
        r = np.array([pos]); q = np.array([1.5])
        n, m, L = 32, 4, 10.0
        g = oracle.spread(r, q, L, n, m, "kaiser_bessel")
        tot = 1.5
        for t in range(3):
            u = n * (pos[t] / L % 1.0)
            c = math.floor(u + 0.5)
            tot *= sum(oracle.phi("kaiser_bessel", m, 2.0, u - (c - m + k)) for k in range(2 * m + 1))
        assert abs(g.sum() - tot) < 1e-13 * abs(tot)
        assert np.count_nonzero(g) <= (2 * m + 1) ** 3


def test_spread_layout_x_fastest(oracle):
    """A particle displaced along x only moves weight along the last grid axis [z,y,x]."""
    n, m, L = 32, 4, 32.0
    g = oracle.spread(np.array([[10.0, 16.0, 20.0]]), np.array([1.0]), L, n, m, "gaussian")
    z, y, x = np.unravel_index(np.argmax(g), g.shape)
    assert (x, y, z) == (10, 16, 20)


@pytest.mark.parametrize("window,m,tol", [("kaiser_bessel", 6, 5e-11), ("kaiser_bessel", 4, 5e-7),
                                          ("gaussian", 4, 5e-4)])
def test_Stilde_matches_direct_S_mode_by_mode(oracle, window, m, tol):
    w = make_workload("cfg1")
    out = oracle.enuf(w.r, w.q, w.L, w.alpha, w.k_cut, w.n, m, window, forces=False, want_S=True)
    ml = oracle.modes(w.k_cut)
    S = oracle.direct_S(w.r, w.q, w.L, ml)
    assert np.abs(out["S"] - S).max() < tol * np.abs(S).max()


def test_dft_and_fft_paths_agree(oracle):
    w = make_workload("cfg1")
    a = oracle.enuf_workload(w, use_dft=True)
    b = oracle.enuf_workload(w, use_dft=False)
    assert abs(a["E"] - b["E"]) < 1e-13 * abs(a["E"])
    assert np.abs(a["F"] - b["F"]).max() < 1e-12 * np.abs(a["F"]).max()


# ----------------------------------------------------------------- Oracle B: accuracy

def _rel_rms(a, b):
    return math.sqrt(((a - b) ** 2).sum() / (b ** 2).sum())


def test_error_falls_with_m(oracle):
    """for fixed sigma_s > 1 the error decays rapidly with m."""
    w = make_workload("cfg1")
    Ea, Fa = oracle.direct(w.r, w.q, w.L, w.alpha, w.k_cut)
    for window, bounds in (("gaussian", (5e-3, 2e-5, 2e-7)), ("kaiser_bessel", (3e-3, 3e-7, 1e-10))):
        errs = []
        for m in (2, 4, 6):
            out = oracle.enuf(w.r, w.q, w.L, w.alpha, w.k_cut, w.n, m, window, variant="ik")
            errs.append(_rel_rms(out["F"], Fa))
            assert abs(out["E"] - Ea) / abs(Ea) < bounds[(m - 2) // 2]
        assert errs[0] > 20 * errs[1] > 400 * errs[2]
        assert all(e < b for e, b in zip(errs, bounds))


CASES = [("gaussian", 4, "ik", 3e-5), ("gaussian", 4, "analytic", 3e-4),
         ("gaussian", 6, "ik", 3e-7), ("gaussian", 6, "analytic", 3e-6),
         ("kaiser_bessel", 4, "ik", 5e-7), ("kaiser_bessel", 4, "analytic", 3e-5),
         ("kaiser_bessel", 6, "ik", 1e-10), ("kaiser_bessel", 6, "analytic", 5e-9)]


@pytest.mark.parametrize("window,m,variant,tol", CASES)
def test_brute_force_small_N(oracle, window, m, variant, tol):
    """N = 64: every window / force variant against the direct Ewald sum (BASELINE)."""
    L, alpha, kc, n = 6.0, 2.0 * math.pi / 6.0, 8, 32
    r, q = random_neutral_gas(64, L, seed=123)
    Ea, Fa = oracle.direct(r, q, L, alpha, kc)
    out = oracle.enuf(r, q, L, alpha, kc, n, m, window, variant=variant)
    assert abs(out["E"] - Ea) < tol * abs(Ea)
    assert _rel_rms(out["F"], Fa) < tol


def test_analytic_variant_is_exact_gradient_of_enuf_energy(oracle):
    """the analytic-derivative force is -grad of E~ (step 5) itself."""
    L, alpha, kc, n, m = 6.0, 1.0, 8, 32, 4
    r, q = random_neutral_gas(10, L, seed=321)
    for window in ("gaussian", "kaiser_bessel"):
        F = oracle.enuf(r, q, L, alpha, kc, n, m, window, variant="analytic")["F"]
        h = 1e-5
        for i, d in ((0, 0), (3, 1), (9, 2)):
            rp = r.copy(); rp[i, d] += h
            rm = r.copy(); rm[i, d] -= h
            ep = oracle.enuf(rp, q, L, alpha, kc, n, m, window, forces=False)["E"]
            em = oracle.enuf(rm, q, L, alpha, kc, n, m, window, forces=False)["E"]
            assert abs(F[i, d] + (ep - em) / (2 * h)) < 5e-9 * np.abs(F).max(), (window, i, d)


def test_ik_variant_conserves_momentum(oracle):
    """R16: sum_i F_i = 0 to round-off for the ik variant (and not for the analytic one)."""
    w = make_workload("cfg1")
    F = oracle.enuf_workload(w, variant="ik")["F"]
    assert np.abs(F.sum(0)).max() < 1e-10 * np.abs(F).max()


def test_enuf_invariances(oracle):
    """Translation by a lattice vector, charge scaling (E, F ~ q^2), q = 0 particles inert."""
    L, alpha, kc, n, m = 6.0, 1.0, 8, 32, 4
    r, q = random_neutral_gas(20, L, seed=4)
    a = oracle.enuf(r, q, L, alpha, kc, n, m, "kaiser_bessel")
    b = oracle.enuf(r + np.array([L, -2 * L, 3 * L]), q, L, alpha, kc, n, m, "kaiser_bessel")
    assert abs(a["E"] - b["E"]) < 1e-12 * abs(a["E"])
    assert np.abs(a["F"] - b["F"]).max() < 1e-11 * np.abs(a["F"]).max()
    c = oracle.enuf(r, 3 * q, L, alpha, kc, n, m, "kaiser_bessel")
    assert abs(c["E"] - 9 * a["E"]) < 1e-13 * abs(c["E"])
    assert np.abs(c["F"] - 9 * a["F"]).max() < 1e-12 * np.abs(c["F"]).max()
    r2 = np.vstack([r, [[1.0, 2.0, 3.0]]]); q2 = np.append(q, 0.0)
    d = oracle.enuf(r2, q2, L, alpha, kc, n, m, "kaiser_bessel")
    assert d["E"] == a["E"] and np.array_equal(d["F"][:-1], a["F"]) and not d["F"][-1].any()


@pytest.mark.parametrize("variant", ["analytic", "ik"])
@pytest.mark.parametrize("window,m", [("kaiser_bessel", 6), ("gaussian", 4)])
def test_enuf_sampled_forces_match_full(oracle, variant, window, m):
    """The `sample` branch of orc_gather / orc_enuf (the one the config 4 / 5 parity tests rely on): forces on a
    sample of particles are the rows of the full result, in the sample's order, bit for bit (same E too)."""
    L, alpha, kc, n = 6.0, 1.0, 8, 32
    r, q = random_neutral_gas(40, L, seed=12)
    q[5] = 0.0                                  # a neutral particle in the sample
    sample = [5, 39, 0, 17, 18]
    full = oracle.enuf(r, q, L, alpha, kc, n, m, window, variant=variant, slater_lambda=0.3)
    part = oracle.enuf(r, q, L, alpha, kc, n, m, window, variant=variant, slater_lambda=0.3, sample=sample)
    assert part["F"].shape == (5, 3)
    assert np.array_equal(part["F"], full["F"][sample])
    assert part["E"] == full["E"]
    assert not part["F"][0].any()


def test_slater_factor_against_direct_and_limit(oracle):
    """R19 (unpinned against the paper): Oracle B with the factor vs Oracle A with the factor."""
    L, alpha, kc, n, m, lam = 6.0, 1.0, 8, 32, 6, 0.4
    r, q = random_neutral_gas(30, L, seed=8)
    Ea, Fa = oracle.direct(r, q, L, alpha, kc, slater_lambda=lam)
    out = oracle.enuf(r, q, L, alpha, kc, n, m, "kaiser_bessel", variant="ik", slater_lambda=lam)
    assert abs(out["E"] - Ea) < 1e-10 * abs(Ea) and _rel_rms(out["F"], Fa) < 1e-9
    E0, _ = oracle.direct(r, q, L, alpha, kc, forces=False)
    assert Ea < E0    # smearing lowers every |k| > 0 weight


def test_predicted_error_cfg2(oracle):
    """cfg2 (KB m=6) ENUF vs direct, both variants."""
    w = make_workload("cfg2")
    Ea, Fa = oracle.direct(w.r, w.q, w.L, w.alpha, w.k_cut)
    for variant, tol in (("ik", 5e-10), ("analytic", 5e-9)):
        out = oracle.enuf_workload(w, variant=variant)
        assert abs(out["E"] - Ea) < 1e-10 * abs(Ea)
        assert _rel_rms(out["F"], Fa) < tol


# ------------------------------------------------------------------ Oracle R (real-space part)

def test_real_forces_are_minus_gradient_of_pinned_energy(oracle):
    """Eq. 29 (garbled; reading R24): F_i^R = -dU^R/dr_i, with U^R the real-space
    energy that the Madelung / Wigner pins fix.  Central differences, images included."""
    L, alpha, rc = 3.0, 1.3, 4.0
    r, q = random_neutral_gas(20, L, seed=5)
    e_i, F = oracle.real_forces(r, q, L, alpha, rc, shells=2)
    assert abs(e_i.sum() - oracle.real_energy(r, q, L, alpha, rc, 2)) <= 1e-13 * abs(e_i.sum())
    # cutoff-crossing pairs make U^R discontinuous at the 1e-7 level only if a pair sits within h of r_cut
    h = 1e-5
    for i in (0, 7, 19):
        for t in range(3):
            rp, rm = r.copy(), r.copy()
            rp[i, t] += h; rm[i, t] -= h
            fd = -(oracle.real_energy(rp, q, L, alpha, rc, 2) - oracle.real_energy(rm, q, L, alpha, rc, 2)) / (2 * h)
            assert abs(fd - F[i, t]) <= 2e-7 * np.abs(F).max() + 5e-6 * math.erfc(alpha * rc)


def test_real_forces_newton_third_law_and_two_particles(oracle):
    L, alpha = 10.0, 0.4
    r, q = random_neutral_gas(50, L, seed=9)
    _, F = oracle.real_forces(r, q, L, alpha, L / 2)
    assert np.abs(F.sum(axis=0)).max() <= 1e-13 * np.abs(F).max()
    # two opposite charges at distance d along x: F_0 = -q^2 [erfc(a d)/d^2 + 2a/sqrt(pi) exp(-a^2 d^2)/d] (attractive)
    d = 1.7
    r2 = np.array([[1.0, 2.0, 3.0], [1.0 + d, 2.0, 3.0]]); q2 = np.array([1.0, -1.0])
    e2, F2 = oracle.real_forces(r2, q2, L, alpha, 4.0)
    mag = math.erfc(alpha * d) / d ** 2 + 2 * alpha / math.sqrt(math.pi) * math.exp(-(alpha * d) ** 2) / d
    assert F2[0, 0] == pytest.approx(mag, rel=1e-14) and F2[1, 0] == pytest.approx(-mag, rel=1e-14)
    assert np.abs(F2[:, 1:]).max() == 0.0
    assert e2.sum() == pytest.approx(-math.erfc(alpha * d) / d, rel=1e-14)


def test_real_forces_sample_matches_full(oracle):
    L, alpha = 6.0, 0.8
    r, q = random_neutral_gas(64, L, seed=3)
    e, F = oracle.real_forces(r, q, L, alpha, 3.0)
    es, Fs = oracle.real_forces(r, q, L, alpha, 3.0, sample=[5, 0, 63])
    assert np.array_equal(Fs, F[[5, 0, 63]]) and np.array_equal(es, e[[5, 0, 63]])


def test_slater_real_space_factors(oracle):
    """Eq. 57-60: B_U/r -> 1/lambda and B_F -> 0 as r -> 0; B_U, B_F -> 1 at large r;
    Eq. 53 -> 54: -d/dr [B_U(r)/r] = B_F(r)/r^2 (central differences); lambda = 0 is the point charge."""
    lam = 0.25
    for d in (1e-6, 1e-5):
        assert oracle.slater_BU(d, lam) / d == pytest.approx(1.0 / lam, rel=1e-4)
        assert abs(oracle.slater_BF(d, lam)) < 1e-8
    assert oracle.slater_BU(40 * lam, lam) == pytest.approx(1.0, abs=1e-30 + 1e-15)
    assert oracle.slater_BF(40 * lam, lam) == pytest.approx(1.0, abs=1e-15)
    assert oracle.slater_BU(0.7, 0.0) == 1.0 and oracle.slater_BF(0.7, 0.0) == 1.0
    h = 1e-6
    for d in (0.05, 0.2, 0.6, 1.5):
        dU = (oracle.slater_BU(d + h, lam) / (d + h) - oracle.slater_BU(d - h, lam) / (d - h)) / (2 * h)
        assert -dU == pytest.approx(oracle.slater_BF(d, lam) / d ** 2, rel=2e-8)
    # beta = R_c/lambda = 1.125: B_U, B_F "converge to unity when r >= 3.0 R_c" (:463): 0.5 % and 3.6 % off
    assert abs(oracle.slater_BU(3.0, 1 / 1.125) - 1) < 1e-2 and abs(oracle.slater_BF(3.0, 1 / 1.125) - 1) < 5e-2
    # in the pair sum the factors multiply the energy and force terms (two particles, alpha -> 0: erfc -> 1)
    r2 = np.array([[0.0, 0.0, 0.0], [0.3, 0.0, 0.0]]); q2 = np.array([1.0, 1.0])
    e2, F2 = oracle.real_forces(r2, q2, 50.0, 1e-9, 1.0, slater_lambda=lam)
    assert e2.sum() == pytest.approx(oracle.slater_BU(0.3, lam) / 0.3, rel=1e-8)
    assert F2[1, 0] == pytest.approx(oracle.slater_BF(0.3, lam) / 0.09, rel=1e-8)


# ----------------------------------------------------------------- orthorhombic boxes

def _box_gas(N, Lb, seed):
    rng = np.random.default_rng(seed)
    r = rng.uniform(0.0, 1.0, size=(N, 3)) * np.asarray(Lb)
    q = np.where(np.arange(N) % 2 == 0, 1.0, -1.0) * (1.0 + 0.2 * rng.uniform(size=N))
    q -= q.mean()
    return r, q


def test_box_with_equal_edges_is_the_cubic_case(oracle):
    L, alpha, kc, n, m = 5.0, 1.2, 7, 32, 3
    r, q = random_neutral_gas(20, L, seed=11)
    Lb = [L, L, L]
    assert np.array_equal(oracle.modes_box(kc, Lb), oracle.modes(kc))
    Ea, Fa = oracle.direct(r, q, L, alpha, kc, slater_lambda=0.3)
    Eb, Fb = oracle.direct_box(r, q, Lb, alpha, kc, slater_lambda=0.3)
    assert abs(Ea - Eb) <= 1e-13 * abs(Ea) and np.abs(Fa - Fb).max() <= 1e-13 * np.abs(Fa).max()
    for variant in ("analytic", "ik"):
        a = oracle.enuf(r, q, L, alpha, kc, n, m, "kaiser_bessel", variant=variant, want_S=True)
        b = oracle.enuf_box(r, q, Lb, alpha, kc, n, m, "kaiser_bessel", variant=variant, want_S=True)
        assert abs(a["E"] - b["E"]) <= 1e-13 * abs(a["E"])
        assert np.abs(a["F"] - b["F"]).max() <= 1e-13 * np.abs(a["F"]).max()
        assert np.abs(a["S"] - b["S"]).max() <= 1e-13 * np.abs(a["S"]).max()


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_box_supercell_doubles_the_energy(oracle, axis):
    """A cubic cell repeated once along one axis is the same crystal: the box (2L, L, L) with k_cut doubled
    holds exactly the cubic wave vectors (odd indices along the long axis have S = 0), so E doubles and
    every copy feels the cubic forces.  Fixes the per-direction scaling of h, V and the cutoff set."""
    L, alpha, kc = 4.0, 1.3, 5
    r, q = random_neutral_gas(14, L, seed=21 + axis)
    Ec, Fc = oracle.direct(r, q, L, alpha, kc)
    Lb = [L, L, L]; Lb[axis] = 2 * L
    shift = np.zeros(3); shift[axis] = L
    r2 = np.concatenate([r, r + shift]); q2 = np.concatenate([q, q])
    Eb, Fb = oracle.direct_box(r2, q2, Lb, alpha, 2 * kc)
    assert abs(Eb - 2 * Ec) <= 1e-12 * abs(Ec)
    assert np.abs(Fb[:14] - Fc).max() <= 1e-12 * np.abs(Fc).max()
    assert np.abs(Fb[14:] - Fc).max() <= 1e-12 * np.abs(Fc).max()
    # the mode set: n_axis even <-> a cubic mode; the count of modes with S != 0 is the cubic count
    mb = oracle.modes_box(2 * kc, Lb)
    even = mb[mb[:, axis] % 2 == 0].copy(); even[:, axis] //= 2
    assert sorted(map(tuple, even)) == sorted(map(tuple, oracle.modes(kc)))


def test_box_direct_forces_are_minus_gradient(oracle):
    Lb = [3.0, 4.5, 6.1]
    r, q = _box_gas(12, Lb, seed=3)
    alpha, kc = 1.4, 9
    _, F = oracle.direct_box(r, q, Lb, alpha, kc, slater_lambda=0.2)
    h = 1e-5
    for i in (0, 4, 11):
        for d in range(3):
            rp = r.copy(); rp[i, d] += h
            rm = r.copy(); rm[i, d] -= h
            ep, _ = oracle.direct_box(rp, q, Lb, alpha, kc, slater_lambda=0.2, forces=False)
            em, _ = oracle.direct_box(rm, q, Lb, alpha, kc, slater_lambda=0.2, forces=False)
            assert abs(F[i, d] + (ep - em) / (2 * h)) < 2e-9 * np.abs(F).max()
    assert np.abs(F.sum(axis=0)).max() < 1e-12 * np.abs(F).max()


def test_box_total_energy_independent_of_alpha(oracle):
    """Real + reciprocal - self of a box does not depend on the splitting parameter: the real-space sum is done
    here in numpy over image shells (erfc(alpha d)/d, Eq. 17) -- pins exp(-pi^2 h^2/alpha^2)/h^2 and 1/(2 pi V)."""
    from scipy.special import erfc
    Lb = np.array([3.0, 3.6, 4.4])
    r, q = _box_gas(8, Lb, seed=9)
    tot = []
    for alpha, kc in ((1.6, 14), (2.0, 17)):
        e_rec, _ = oracle.direct_box(r, q, Lb, alpha, kc, forces=False)
        e_real = 0.0
        for ix in range(-2, 3):
            for iy in range(-2, 3):
                for iz in range(-2, 3):
                    sh = np.array([ix, iy, iz]) * Lb
                    d = np.linalg.norm(r[:, None, :] - r[None, :, :] + sh, axis=2)
                    qq = q[:, None] * q[None, :]
                    if ix == iy == iz == 0:
                        np.fill_diagonal(d, np.inf)
                    e_real += 0.5 * (qq * erfc(alpha * d) / d).sum()
        tot.append(e_real + e_rec - alpha / math.sqrt(math.pi) * (q ** 2).sum())
    assert abs(tot[0] - tot[1]) < 1e-9 * abs(tot[0])


@pytest.mark.parametrize("variant,bound", [("analytic", 2e-7), ("ik", 2e-7)])
def test_box_enuf_against_direct(oracle, variant, bound):
    Lb = [5.0, 6.5, 8.0]
    r, q = _box_gas(40, Lb, seed=17)
    alpha, kc, n, m = 1.0, 8, 32, 6
    Ea, Fa = oracle.direct_box(r, q, Lb, alpha, kc)
    b = oracle.enuf_box(r, q, Lb, alpha, kc, n, m, "kaiser_bessel", variant=variant, want_S=True)
    assert abs(b["E"] - Ea) <= bound * abs(Ea)
    assert np.abs(b["F"] - Fa).max() <= bound * np.abs(Fa).max()
    # S~ mode by mode in modes_box order
    ml = oracle.modes_box(kc, Lb)
    x = r / np.asarray(Lb)
    S = (q[None, :] * np.exp(-2j * np.pi * (ml @ x.T))).sum(axis=1)
    assert np.abs(b["S"] - S).max() <= bound * np.abs(S).max()


def test_box_analytic_variant_is_exact_gradient(oracle):
    Lb = [4.0, 5.0, 7.0]
    r, q = _box_gas(10, Lb, seed=5)
    alpha, kc, n, m = 1.1, 7, 32, 3
    F = oracle.enuf_box(r, q, Lb, alpha, kc, n, m, "gaussian", variant="analytic")["F"]
    h = 1e-5
    for i, d in ((0, 0), (3, 1), (9, 2), (5, 0), (5, 2)):
        rp = r.copy(); rp[i, d] += h
        rm = r.copy(); rm[i, d] -= h
        ep = oracle.enuf_box(rp, q, Lb, alpha, kc, n, m, "gaussian", forces=False)["E"]
        em = oracle.enuf_box(rm, q, Lb, alpha, kc, n, m, "gaussian", forces=False)["E"]
        assert abs(F[i, d] + (ep - em) / (2 * h)) < 5e-9 * np.abs(F).max(), (i, d)
