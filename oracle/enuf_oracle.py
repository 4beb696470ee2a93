"""ctypes binding of oracle/enuf_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this.  It never imports the CUDA package.  ``build()`` compiles the C file with
gcc (portable flags: the .so travels from the build box to the GPU box).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "enuf_oracle.c")
_LIB = os.path.join(_HERE, "libenuf_oracle.so")

WINDOWS = {"gaussian": 0, "kaiser_bessel": 1, "bspline": 2, "sinc_power": 3}
VARIANTS = {"analytic": 0, "ik": 1}

_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle shared library if missing or older than its source."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    cmd = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
           "-D_DEFAULT_SOURCE", "-o", _LIB, _SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return _LIB


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double)) if a is not None else None


def _f64(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        d, i, i64, p = C.c_double, C.c_int, C.c_int64, C.POINTER(C.c_double)
        pi32, pi64 = C.POINTER(C.c_int), C.POINTER(C.c_int64)
        L.orc_num_threads.restype = i
        L.orc_set_threads.argtypes = [i]
        for name in ("orc_phi", "orc_dphi"):
            f = getattr(L, name); f.restype = d; f.argtypes = [i, i, d, d]
        L.orc_Phi.restype = d; L.orc_Phi.argtypes = [i, i, d, i, i]
        L.orc_w.restype = d; L.orc_w.argtypes = [i, d, d]
        L.orc_slater_f2.restype = d; L.orc_slater_f2.argtypes = [i, d, d]
        L.orc_ncut.restype = i; L.orc_ncut.argtypes = [d, d, d]
        L.orc_alpha_from_rc.restype = d; L.orc_alpha_from_rc.argtypes = [d, d]
        L.orc_slater_BU.restype = d; L.orc_slater_BU.argtypes = [d, d]
        L.orc_slater_BF.restype = d; L.orc_slater_BF.argtypes = [d, d]
        L.orc_real_forces.restype = None
        L.orc_real_forces.argtypes = [i64, p, p, d, d, d, i, d, i64, pi64, p, p]
        L.orc_direct_S.restype = None
        L.orc_direct_S.argtypes = [i64, p, p, d, i64, pi32, p, p]
        L.orc_modes.restype = i64; L.orc_modes.argtypes = [i, pi32]
        L.orc_direct.restype = i
        L.orc_direct.argtypes = [i64, p, p, d, d, i, d, p, p, i64, pi64]
        L.orc_real_energy.restype = d; L.orc_real_energy.argtypes = [i64, p, p, d, d, d, i]
        L.orc_self_energy.restype = d; L.orc_self_energy.argtypes = [i64, p, d]
        L.orc_spread.restype = None; L.orc_spread.argtypes = [i64, p, p, d, i, i, i, d, p]
        L.orc_fft_line.restype = None; L.orc_fft_line.argtypes = [i, i, i, p, p]
        L.orc_fft3d.restype = None; L.orc_fft3d.argtypes = [i, i, i, p, p]
        L.orc_scale.restype = d
        L.orc_scale.argtypes = [i, i, d, d, d, i, i, d, p, p, i, p, p, p, p]
        L.orc_gather.restype = None
        L.orc_gather.argtypes = [i64, p, p, d, i, i, i, d, i, p, p, i64, pi64]
        L.orc_enuf.restype = i
        L.orc_enuf.argtypes = [i64, p, p, d, d, i, i, i, i, d, i, d, i, p, p, i64, pi64, p, p, p]
        # orthorhombic boxes (Lb = three edges)
        L.orc_box_s.restype = d; L.orc_box_s.argtypes = [p, i, i, i]
        L.orc_box_fw.restype = d; L.orc_box_fw.argtypes = [p, d, d, d]
        L.orc_modes_box.restype = i64; L.orc_modes_box.argtypes = [i, p, pi32]
        L.orc_direct_box.restype = i
        L.orc_direct_box.argtypes = [i64, p, p, p, d, i, d, p, p, i64, pi64]
        L.orc_spread_box.restype = None; L.orc_spread_box.argtypes = [i64, p, p, p, i, i, i, d, p]
        L.orc_enuf_box.restype = i
        L.orc_enuf_box.argtypes = [i64, p, p, p, d, i, i, i, i, d, i, d, i, p, p, i64, pi64, p, p, p]
        _lib = L
    return _lib


def num_threads() -> int:
    return lib().orc_num_threads()


def set_threads(t: int) -> None:
    lib().orc_set_threads(int(t))


def phi(window, m, sigma, d):
    return lib().orc_phi(WINDOWS[window], m, sigma, float(d))


def dphi(window, m, sigma, d):
    return lib().orc_dphi(WINDOWS[window], m, sigma, float(d))


def Phi(window, m, sigma, n, k):
    return lib().orc_Phi(WINDOWS[window], m, sigma, n, int(k))


def w(n2, alpha, L):
    return lib().orc_w(int(n2), alpha, L)


def slater_f2(n2, lam, L):
    return lib().orc_slater_f2(int(n2), lam, L)


def ncut(alpha, L, delta):
    return lib().orc_ncut(alpha, L, delta)


def alpha_from_rc(r_c, delta):
    return lib().orc_alpha_from_rc(r_c, delta)


def modes(k_cut):
    """All n in K = {0 < |n|^2 <= k_cut^2} as an (|K|, 3) int32 array (fixed order)."""
    nk = lib().orc_modes(k_cut, None)
    out = np.empty((nk, 3), dtype=np.int32)
    lib().orc_modes(k_cut, out.ctypes.data_as(C.POINTER(C.c_int)))
    return out


def direct_S(r, q, L, mode_list):
    r, q = _f64(r), _f64(q)
    ml = np.ascontiguousarray(np.asarray(mode_list, dtype=np.int32).reshape(-1, 3))
    sr = np.empty(ml.shape[0]); si = np.empty(ml.shape[0])
    lib().orc_direct_S(q.shape[0], _dp(r), _dp(q), L, ml.shape[0],
                       ml.ctypes.data_as(C.POINTER(C.c_int)), _dp(sr), _dp(si))
    return sr + 1j * si


def direct(r, q, L, alpha, k_cut, slater_lambda=0.0, forces=True, sample=None):
    """Oracle A: (E_rec, F) by the direct O(N|K|) sum. F is (N,3) or (len(sample),3)."""
    r, q = _f64(r), _f64(q)
    N = q.shape[0]
    E = C.c_double(0.0)
    F = None
    ns, sp = 0, None
    if sample is not None:
        sample = np.ascontiguousarray(np.asarray(sample, dtype=np.int64))
        ns, sp = sample.shape[0], sample.ctypes.data_as(C.POINTER(C.c_int64))
    if forces:
        F = np.zeros((ns if ns else N, 3))
    rc = lib().orc_direct(N, _dp(r), _dp(q), L, alpha, k_cut, slater_lambda, C.byref(E),
                          _dp(F), ns, sp)
    if rc:
        raise MemoryError("orc_direct failed")
    return E.value, F


def real_energy(r, q, L, alpha, r_cut, shells=1):
    r, q = _f64(r), _f64(q)
    return lib().orc_real_energy(q.shape[0], _dp(r), _dp(q), L, alpha, r_cut, shells)


def slater_BU(d, lam):
    return lib().orc_slater_BU(float(d), float(lam))


def slater_BF(d, lam):
    return lib().orc_slater_BF(float(d), float(lam))


def real_forces(r, q, L, alpha, r_cut, shells=1, slater_lambda=0.0, sample=None):
    """Oracle R: real-space Ewald part. Returns (e_i, F) for all particles or for `sample`;
    e_i = 1/2 q_i sum_j q_j B_U erfc(alpha d)/d, so e_i summed over ALL particles is E_real."""
    r, q = _f64(r), _f64(q)
    N = q.shape[0]
    ns, sp = 0, None
    if sample is not None:
        sample = np.ascontiguousarray(np.asarray(sample, dtype=np.int64))
        ns, sp = sample.shape[0], sample.ctypes.data_as(C.POINTER(C.c_int64))
    cnt = ns if ns else N
    F = np.zeros((cnt, 3)); e = np.zeros(cnt)
    lib().orc_real_forces(N, _dp(r), _dp(q), L, alpha, r_cut, shells, slater_lambda, ns, sp, _dp(F), _dp(e))
    return e, F


def self_energy(q, alpha):
    q = _f64(q)
    return lib().orc_self_energy(q.shape[0], _dp(q), alpha)


def spread(r, q, L, n, m, window, sigma=2.0):
    r, q = _f64(r), _f64(q)
    g = np.zeros((n, n, n))
    lib().orc_spread(q.shape[0], _dp(r), _dp(q), L, n, m, WINDOWS[window], sigma, _dp(g))
    return g


def fft_line(x, sign, use_dft):
    x = np.asarray(x, dtype=np.complex128)
    re = np.ascontiguousarray(x.real); im = np.ascontiguousarray(x.imag)
    lib().orc_fft_line(x.shape[0], sign, int(use_dft), _dp(re), _dp(im))
    return re + 1j * im


def fft3d(a, sign, use_dft=False):
    a = np.asarray(a, dtype=np.complex128)
    n = a.shape[0]
    re = np.ascontiguousarray(a.real); im = np.ascontiguousarray(a.imag)
    lib().orc_fft3d(n, sign, int(use_dft), _dp(re), _dp(im))
    return re + 1j * im


def enuf(r, q, L, alpha, k_cut, n, m, window, sigma=2.0, variant="analytic",
         slater_lambda=0.0, use_dft=False, forces=True, sample=None,
         want_grid=False, want_S=False):
    """Oracle B. Returns dict(E, F, grid, S) (absent outputs are None).

    S is S~ over ``modes(k_cut)`` in that order; grid is the (n,n,n) spread grid [z,y,x].
    """
    r, q = _f64(r), _f64(q)
    N = q.shape[0]
    E = C.c_double(0.0)
    ns, sp = 0, None
    if sample is not None:
        sample = np.ascontiguousarray(np.asarray(sample, dtype=np.int64))
        ns, sp = sample.shape[0], sample.ctypes.data_as(C.POINTER(C.c_int64))
    F = np.zeros((ns if ns else N, 3)) if forces else None
    grid = np.zeros((n, n, n)) if want_grid else None
    sr = si = None
    if want_S:
        nk = lib().orc_modes(k_cut, None)
        sr = np.empty(nk); si = np.empty(nk)
    rc = lib().orc_enuf(N, _dp(r), _dp(q), L, alpha, k_cut, n, m, WINDOWS[window], sigma,
                        VARIANTS[variant], slater_lambda, int(use_dft), C.byref(E), _dp(F),
                        ns, sp, _dp(grid), _dp(sr), _dp(si))
    if rc:
        raise RuntimeError(f"orc_enuf failed with code {rc}")
    return {"E": E.value, "F": F, "grid": grid,
            "S": (sr + 1j * si) if want_S else None}


def enuf_workload(w, variant="analytic", **kw):
    """Oracle B on an enuf_inputs.Workload (inputs promoted exactly to fp64)."""
    return enuf(w.r, w.q, w.L, w.alpha, w.k_cut, w.n, w.m, w.window, w.sigma,
                variant=variant, slater_lambda=w.slater_lambda, **kw)


# ------------------------------------------------------------------ orthorhombic boxes

def _box(Lb):
    Lb = _f64(Lb).reshape(3)
    return Lb


def modes_box(k_cut, Lb):
    """All n in K = {n != 0 : |h| Lmax <= k_cut}, h = n / Lb, as an (|K|, 3) int32 array (fixed order)."""
    Lb = _box(Lb)
    nk = lib().orc_modes_box(k_cut, _dp(Lb), None)
    out = np.empty((nk, 3), dtype=np.int32)
    lib().orc_modes_box(k_cut, _dp(Lb), out.ctypes.data_as(C.POINTER(C.c_int)))
    return out


def direct_box(r, q, Lb, alpha, k_cut, slater_lambda=0.0, forces=True, sample=None):
    """Oracle A for a box with edges Lb: (E_rec, F)."""
    r, q, Lb = _f64(r), _f64(q), _box(Lb)
    N = q.shape[0]
    E = C.c_double(0.0)
    F = None
    ns, sp = 0, None
    if sample is not None:
        sample = np.ascontiguousarray(np.asarray(sample, dtype=np.int64))
        ns, sp = sample.shape[0], sample.ctypes.data_as(C.POINTER(C.c_int64))
    if forces:
        F = np.zeros((ns if ns else N, 3))
    rc = lib().orc_direct_box(N, _dp(r), _dp(q), _dp(Lb), alpha, k_cut, slater_lambda, C.byref(E),
                              _dp(F), ns, sp)
    if rc:
        raise MemoryError("orc_direct_box failed")
    return E.value, F


def spread_box(r, q, Lb, n, m, window, sigma=2.0):
    r, q, Lb = _f64(r), _f64(q), _box(Lb)
    g = np.zeros((n, n, n))
    lib().orc_spread_box(q.shape[0], _dp(r), _dp(q), _dp(Lb), n, m, WINDOWS[window], sigma, _dp(g))
    return g


def enuf_box(r, q, Lb, alpha, k_cut, n, m, window, sigma=2.0, variant="analytic",
             slater_lambda=0.0, use_dft=False, forces=True, sample=None, want_grid=False, want_S=False):
    """Oracle B for a box with edges Lb; same returns as enuf(), S over modes_box(k_cut, Lb)."""
    r, q, Lb = _f64(r), _f64(q), _box(Lb)
    N = q.shape[0]
    E = C.c_double(0.0)
    ns, sp = 0, None
    if sample is not None:
        sample = np.ascontiguousarray(np.asarray(sample, dtype=np.int64))
        ns, sp = sample.shape[0], sample.ctypes.data_as(C.POINTER(C.c_int64))
    F = np.zeros((ns if ns else N, 3)) if forces else None
    grid = np.zeros((n, n, n)) if want_grid else None
    sr = si = None
    if want_S:
        nk = lib().orc_modes_box(k_cut, _dp(Lb), None)
        sr = np.empty(nk); si = np.empty(nk)
    rc = lib().orc_enuf_box(N, _dp(r), _dp(q), _dp(Lb), alpha, k_cut, n, m, WINDOWS[window], sigma,
                            VARIANTS[variant], slater_lambda, int(use_dft), C.byref(E), _dp(F),
                            ns, sp, _dp(grid), _dp(sr), _dp(si))
    if rc:
        raise RuntimeError(f"orc_enuf_box failed with code {rc}")
    return {"E": E.value, "F": F, "grid": grid, "S": (sr + 1j * si) if want_S else None}
