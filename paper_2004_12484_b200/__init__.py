"""Python binding of libenuf_b200.so (include/enuf.h) -- argument marshalling only.

Every step of the ENUF reciprocal-space path (bin, spread, FFT, scale, inverse FFT,
gather, energy) runs in the library's CUDA kernels; PyTorch supplies device memory and the
CUDA stream.  There is no CPU fallback: importing works without a GPU (so the symbol test
can run), but any compute call without a CUDA device raises ``EnufError``.

    import torch, paper_2004_12484_b200 as enuf
    plan = enuf.Plan(N, L, alpha, k_cut, M, sigma=2.0, m=6, dtype=torch.float32)
    E, F = plan.energy_forces(r, q)          # r (N,3), q (N,) CUDA tensors
"""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libenuf_b200.so")

OK, EINVAL, ENOMEM, ECUDA, ESTATE = 0, -1, -2, -3, -4
OPT_PRECISION, OPT_WINDOW, OPT_FORCE_VARIANT, OPT_SLATER_LAMBDA = 1, 2, 3, 4
OPT_NUM_PARTICLES, OPT_PROFILE, OPT_KEEP_SPECTRUM, OPT_SPREAD_ZCHUNK = 5, 6, 7, 8
OPT_PDL = 10
OPT_SPREAD_SPARSE = 11
OPT_CUDA_GRAPH = 9
F32, F64 = 0, 1
WINDOWS = {"gaussian": 0, "kaiser_bessel": 1, "bspline": 2, "sinc_power": 3}
VARIANTS = {"analytic": 0, "ik": 1}
STAGES = ("bin", "spread", "fft", "gather", "energy")

# every symbol include/enuf.h declares (checked by tests/test_abi.py)
SYMBOLS = (
    "enuf_plan_create", "enuf_plan_set", "enuf_plan_set_stream", "enuf_energy_forces",
    "enuf_energy_forces_host", "enuf_plan_energy", "enuf_plan_stage_ms", "enuf_plan_stage_ms_mean",
    "enuf_plan_launch_count",
    "enuf_spectrum_partial", "enuf_plan_spectrum_buffer", "enuf_forces_from_spectrum",
    "enuf_real_space",
    "enuf_plan_copy_field", "enuf_plan_structure_factor", "enuf_spread_only",
    "enuf_plan_workspace_bytes", "enuf_plan_destroy", "enuf_last_error",
    "enuf_ncut", "enuf_alpha_from_rc", "enuf_rc_from_ncut",
    "enuf_plan_create_auto", "enuf_plan_get", "enuf_plan_create_box", "enuf_self_energy_static",
    "enuf_spread_split_check",
)
SELF_STATIC_MAX_N = 1 << 24
GET_ALPHA, GET_K_CUT, GET_M, GET_GRID, GET_SUPPORT = 1, 2, 3, 4, 5


class EnufError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__(f"enuf error {code}: {message}")
        self.code = code


_lib = None


def lib():
    """Load the C-ABI library; fails loudly if it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(
                f"{LIB_PATH} is missing: build it with `python -m paper_2004_12484_b200.build` "
                "(or __graft_entry__.build()). There is no fallback implementation.")
        L = C.CDLL(LIB_PATH)
        vp, d, i, i64 = C.c_void_p, C.c_double, C.c_int, C.c_int64
        L.enuf_plan_create.restype = i
        L.enuf_plan_create.argtypes = [C.POINTER(vp), i64, d, d, i, i, d, i]
        L.enuf_plan_set.restype = i; L.enuf_plan_set.argtypes = [vp, i, d]
        L.enuf_plan_set_stream.restype = i; L.enuf_plan_set_stream.argtypes = [vp, vp]
        L.enuf_energy_forces.restype = i
        L.enuf_energy_forces.argtypes = [vp, vp, vp, vp, C.POINTER(d)]
        L.enuf_energy_forces_host.restype = i
        L.enuf_energy_forces_host.argtypes = [vp, vp, vp, vp, C.POINTER(d)]
        L.enuf_plan_energy.restype = i; L.enuf_plan_energy.argtypes = [vp, C.POINTER(d)]
        L.enuf_real_space.restype = i
        L.enuf_real_space.argtypes = [vp, vp, vp, d, i, vp, C.POINTER(d), C.POINTER(d)]
        L.enuf_spectrum_partial.restype = i; L.enuf_spectrum_partial.argtypes = [vp, vp, vp, vp]
        L.enuf_plan_spectrum_buffer.restype = i
        L.enuf_plan_spectrum_buffer.argtypes = [vp, C.POINTER(vp), C.POINTER(C.c_size_t)]
        L.enuf_forces_from_spectrum.restype = i; L.enuf_forces_from_spectrum.argtypes = [vp, vp, C.POINTER(d)]
        L.enuf_plan_stage_ms.restype = i; L.enuf_plan_stage_ms.argtypes = [vp, C.POINTER(C.c_float), i]
        L.enuf_plan_stage_ms_mean.restype = i
        L.enuf_plan_stage_ms_mean.argtypes = [vp, C.POINTER(C.c_float), i, C.POINTER(i)]
        L.enuf_plan_launch_count.restype = i; L.enuf_plan_launch_count.argtypes = [vp]
        L.enuf_plan_copy_field.restype = i; L.enuf_plan_copy_field.argtypes = [vp, vp]
        L.enuf_plan_structure_factor.restype = i
        L.enuf_plan_structure_factor.argtypes = [vp, i64, C.POINTER(i), C.POINTER(d)]
        L.enuf_spread_only.restype = i; L.enuf_spread_only.argtypes = [vp, vp, vp, vp]
        L.enuf_plan_workspace_bytes.restype = C.c_size_t; L.enuf_plan_workspace_bytes.argtypes = [vp]
        L.enuf_plan_destroy.restype = None; L.enuf_plan_destroy.argtypes = [vp]
        L.enuf_last_error.restype = C.c_char_p; L.enuf_last_error.argtypes = []
        L.enuf_ncut.restype = i; L.enuf_ncut.argtypes = [d, d, d]
        L.enuf_alpha_from_rc.restype = d; L.enuf_alpha_from_rc.argtypes = [d, d]
        L.enuf_rc_from_ncut.restype = d; L.enuf_rc_from_ncut.argtypes = [i, d, d]
        L.enuf_plan_create_box.restype = i
        L.enuf_plan_create_box.argtypes = [C.POINTER(vp), i64, C.POINTER(d), d, i, i, d, i]
        L.enuf_plan_create_auto.restype = i
        L.enuf_plan_create_auto.argtypes = [C.POINTER(vp), i64, d, d, d, d, i]
        L.enuf_plan_get.restype = i; L.enuf_plan_get.argtypes = [vp, i, C.POINTER(d)]
        L.enuf_spread_split_check.restype = i
        L.enuf_spread_split_check.argtypes = [i, i, i, i, i, i, C.POINTER(i), C.POINTER(i), C.POINTER(i)]
        L.enuf_self_energy_static.restype = i
        L.enuf_self_energy_static.argtypes = [vp, i64, i, d, vp, vp]
        _lib = L
    return _lib


def _check(code: int) -> None:
    if code != OK:
        raise EnufError(code, lib().enuf_last_error().decode())


def ncut(alpha: float, L: float, delta: float) -> int:
    """Eq. 31: smallest integer n_c >= (alpha L/pi) sqrt(-ln delta)."""
    return lib().enuf_ncut(alpha, L, delta)


def alpha_from_rc(r_c: float, delta: float) -> float:
    """Eq. 32 read as exp(-alpha^2 r_c^2) = delta."""
    return lib().enuf_alpha_from_rc(r_c, delta)


def rc_from_ncut(n_c: int, alpha: float, L: float) -> float:
    """Eq. 32: r_c = pi n_c / (alpha^2 L)."""
    return lib().enuf_rc_from_ncut(n_c, alpha, L)


def shard_bounds(N: int, rank: int, world: int):
    """[lo, hi) of the particles rank `rank` of `world` owns when N particles are split by index
    into contiguous, near-equal shards (HP-ENUF partitions by particle)."""
    if not (0 <= rank < world):
        raise ValueError("rank must be in [0, world)")
    base, rem = divmod(int(N), int(world))
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def all_reduce_sum_(t, group=None):
    """In-place sum of a tensor over the ranks of `group` (identity without an initialised
    process group or with one rank): the one exchange step of the sharded path."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return t


class _DeviceBuffer:
    """A plan-owned device buffer exposed through __cuda_array_interface__ (no copy)."""

    def __init__(self, ptr: int, count: int, typestr: str):
        self.__cuda_array_interface__ = {"shape": (count,), "typestr": typestr, "data": (ptr, False),
                                         "version": 2, "strides": None}


class Plan:
    """enuf_plan_create (L a number) or enuf_plan_create_box (L = three edges) / enuf_plan_set /
    enuf_energy_forces / enuf_plan_destroy."""

    def __init__(self, N, L, alpha, k_cut, M, sigma=2.0, m=6, dtype=None, window="kaiser_bessel",
                 variant="analytic", slater_lambda=0.0, profile=False, keep_spectrum=False, cuda_graph=False):
        import torch
        self._torch = torch
        self._h = C.c_void_p()
        self.dtype = torch.float32 if dtype is None else dtype
        if self.dtype not in (torch.float32, torch.float64):
            raise ValueError("dtype must be torch.float32 or torch.float64")
        self.N, self.n = int(N), int(round(sigma * M))
        self.k_cut = int(k_cut)
        if hasattr(L, "__len__"):      # (Lx, Ly, Lz): orthorhombic box, enuf_plan_create_box
            if len(L) != 3:
                raise ValueError("L must be a number or three box edges")
            Lb = (C.c_double * 3)(*[float(v) for v in L])
            _check(lib().enuf_plan_create_box(C.byref(self._h), int(N), Lb, float(alpha), int(k_cut),
                                              int(M), float(sigma), int(m)))
        else:
            _check(lib().enuf_plan_create(C.byref(self._h), int(N), float(L), float(alpha), int(k_cut),
                                          int(M), float(sigma), int(m)))
        self.set(OPT_PRECISION, F32 if self.dtype == torch.float32 else F64)
        self.set(OPT_WINDOW, WINDOWS[window])
        self.set(OPT_FORCE_VARIANT, VARIANTS[variant])
        self.set(OPT_SLATER_LAMBDA, slater_lambda)
        self.set(OPT_PROFILE, int(profile))
        self.set(OPT_KEEP_SPECTRUM, int(keep_spectrum))
        if cuda_graph:
            self.set(OPT_CUDA_GRAPH, 1)

    @classmethod
    def auto(cls, N, L, delta, r_c, sigma=2.0, m=6, **kw):
        """enuf_plan_create_auto: alpha, k_cut and M from the accuracy delta and the real-space cutoff r_c by the
        parameter rule Eq. 31-32.  Other keyword arguments as for Plan()."""
        h = C.c_void_p()
        _check(lib().enuf_plan_create_auto(C.byref(h), int(N), float(L), float(delta), float(r_c), float(sigma), int(m)))
        v = C.c_double(0.0)
        got = {}
        for name, key in (("alpha", GET_ALPHA), ("k_cut", GET_K_CUT), ("M", GET_M)):
            _check(lib().enuf_plan_get(h, key, C.byref(v)))
            got[name] = v.value
        lib().enuf_plan_destroy(h)
        return cls(N, L, got["alpha"], int(got["k_cut"]), int(got["M"]), sigma=sigma, m=m, **kw)

    def get(self, key: int) -> float:
        v = C.c_double(0.0)
        _check(lib().enuf_plan_get(self._h, int(key), C.byref(v)))
        return v.value

    @classmethod
    def from_workload(cls, w, **kw):
        import torch
        kw.setdefault("dtype", torch.float64 if w.dtype == "f64" else torch.float32)
        kw.setdefault("window", w.window)
        kw.setdefault("slater_lambda", w.slater_lambda)
        return cls(w.N, w.L, w.alpha, w.k_cut, w.M, sigma=w.sigma, m=w.m, **kw)

    def set(self, key: int, value: float) -> None:
        _check(lib().enuf_plan_set(self._h, int(key), float(value)))

    def set_num_particles(self, N: int) -> None:
        self.set(OPT_NUM_PARTICLES, N)
        self.N = int(N)

    def _use_current_stream(self) -> None:
        s = self._torch.cuda.current_stream().cuda_stream
        _check(lib().enuf_plan_set_stream(self._h, C.c_void_p(s)))

    def _dev(self, t, shape, name):
        torch = self._torch
        if not isinstance(t, torch.Tensor) or not t.is_cuda:
            raise TypeError(f"{name} must be a CUDA tensor")
        if t.dtype != self.dtype or tuple(t.shape) != shape or not t.is_contiguous():
            raise ValueError(f"{name} must be contiguous {self.dtype} of shape {shape}")
        return C.c_void_p(t.data_ptr())

    def energy_forces(self, r, q, F=None, want_energy=True):
        """One evaluation on device tensors. Returns (E or None, F)."""
        torch = self._torch
        if not torch.cuda.is_available():
            raise EnufError(ECUDA, "no CUDA device available; this library has no CPU fallback")
        N = self.N
        if F is None:
            F = torch.empty((N, 3), dtype=self.dtype, device=r.device)
        self._use_current_stream()
        E = C.c_double(0.0)
        _check(lib().enuf_energy_forces(self._h, self._dev(r, (N, 3), "r"), self._dev(q, (N,), "q"),
                                        self._dev(F, (N, 3), "F"), C.byref(E) if want_energy else None))
        return (E.value if want_energy else None), F

    def energy_forces_host(self, r, q=None, F=None):
        """One evaluation on HOST tensors / numpy arrays (H2D and D2H inside the call).  q=None reuses the
        charges of the previous host call, which stay resident on the device."""
        torch = self._torch
        N = self.N
        r_t = r if isinstance(r, torch.Tensor) else torch.from_numpy(r)
        q_t = None if q is None else (q if isinstance(q, torch.Tensor) else torch.from_numpy(q))
        if F is None:
            F = torch.empty((N, 3), dtype=self.dtype)
        for t, shape, name in ((r_t, (N, 3), "r"), (q_t, (N,), "q"), (F, (N, 3), "F")):
            if t is None:
                continue
            if t.is_cuda or t.dtype != self.dtype or tuple(t.shape) != shape or not t.is_contiguous():
                raise ValueError(f"{name} must be a contiguous host {self.dtype} tensor of shape {shape}")
        self._use_current_stream()
        E = C.c_double(0.0)
        _check(lib().enuf_energy_forces_host(self._h, C.c_void_p(r_t.data_ptr()),
                                             C.c_void_p(q_t.data_ptr()) if q_t is not None else None,
                                             C.c_void_p(F.data_ptr()), C.byref(E)))
        return E.value, F

    # ---- sharded evaluation (include/enuf.h, "Sharded evaluation")
    def spectrum_partial(self, r, q, F):
        """a1, a2 and the X, Y forward passes on this rank's particles."""
        N = self.N
        self._use_current_stream()
        _check(lib().enuf_spectrum_partial(self._h, self._dev(r, (N, 3), "r"), self._dev(q, (N,), "q"),
                                           self._dev(F, (N, 3), "F")))

    def spectrum_tensor(self):
        """The plan-owned partial-spectrum buffer as a flat CUDA tensor (a view, no copy): the
        tensor to all-reduce (sum) over ranks between the two halves."""
        torch = self._torch
        ptr, cnt = C.c_void_p(), C.c_size_t(0)
        _check(lib().enuf_plan_spectrum_buffer(self._h, C.byref(ptr), C.byref(cnt)))
        key = (ptr.value, cnt.value)
        if getattr(self, "_spec_key", None) != key:
            buf = _DeviceBuffer(ptr.value, cnt.value, "<f4" if self.dtype == torch.float32 else "<f8")
            self._spec_view = torch.as_tensor(buf, device="cuda")
            self._spec_key = key
        return self._spec_view

    def forces_from_spectrum(self, F, want_energy=True):
        """a4 .. a7 on the (summed) spectrum buffer; forces on this rank's particles."""
        self._use_current_stream()
        E = C.c_double(0.0)
        _check(lib().enuf_forces_from_spectrum(self._h, self._dev(F, (self.N, 3), "F"),
                                               C.byref(E) if want_energy else None))
        return (E.value if want_energy else None), F

    def energy_forces_sharded(self, r, q, F=None, group=None, want_energy=True):
        """One evaluation of a system whose particles are spread over the ranks of `group`
        (each rank passes its own r, q).  Returns (E of the whole system, F of the own particles)."""
        torch = self._torch
        if not torch.cuda.is_available():
            raise EnufError(ECUDA, "no CUDA device available; this library has no CPU fallback")
        if F is None:
            F = torch.empty((self.N, 3), dtype=self.dtype, device=r.device)
        self.spectrum_partial(r, q, F)
        all_reduce_sum_(self.spectrum_tensor(), group)
        return self.forces_from_spectrum(F, want_energy=want_energy)

    def real_space(self, r, q, r_cut, F=None, accumulate=False, want_energy=True):
        """Real-space Ewald part and self term (enuf_real_space). Returns (E_real, E_self, F);
        with accumulate=True the forces are added to F."""
        torch = self._torch
        if not torch.cuda.is_available():
            raise EnufError(ECUDA, "no CUDA device available; this library has no CPU fallback")
        N = self.N
        if F is None:
            if accumulate:
                raise ValueError("accumulate=True needs F")
            F = torch.empty((N, 3), dtype=self.dtype, device=r.device)
        self._use_current_stream()
        Er, Es = C.c_double(0.0), C.c_double(0.0)
        _check(lib().enuf_real_space(self._h, self._dev(r, (N, 3), "r"), self._dev(q, (N,), "q"), float(r_cut),
                                     int(bool(accumulate)), self._dev(F, (N, 3), "F"),
                                     C.byref(Er) if want_energy else None, C.byref(Es) if want_energy else None))
        return (Er.value if want_energy else None), (Es.value if want_energy else None), F

    def energy(self) -> float:
        E = C.c_double(0.0)
        _check(lib().enuf_plan_energy(self._h, C.byref(E)))
        return E.value

    def stage_ms(self) -> dict:
        arr = (C.c_float * len(STAGES))()
        _check(lib().enuf_plan_stage_ms(self._h, arr, len(STAGES)))
        return dict(zip(STAGES, (float(x) for x in arr)))

    def stage_ms_mean(self):
        """(mean per-stage ms, number of evaluations averaged) since profiling was switched on."""
        arr = (C.c_float * len(STAGES))()
        ne = C.c_int(0)
        _check(lib().enuf_plan_stage_ms_mean(self._h, arr, len(STAGES), C.byref(ne)))
        return dict(zip(STAGES, (float(x) for x in arr))), ne.value

    def launch_count(self) -> int:
        return lib().enuf_plan_launch_count(self._h)

    def workspace_bytes(self) -> int:
        return lib().enuf_plan_workspace_bytes(self._h)

    def spread_only(self, r, q):
        """Spread grid g (n,n,n) [z,y,x] as a host tensor (steps a1 + a2)."""
        torch = self._torch
        N, n = self.N, self.n
        out = torch.empty((n, n, n), dtype=self.dtype)
        self._use_current_stream()
        _check(lib().enuf_spread_only(self._h, self._dev(r, (N, 3), "r"), self._dev(q, (N,), "q"),
                                      C.c_void_p(out.data_ptr())))
        return out

    def field(self):
        """Real-space field the gather read (Psi, or B_x for ik), host tensor (n,n,n) [z,y,x]."""
        n = self.n
        out = self._torch.empty((n, n, n), dtype=self.dtype)
        _check(lib().enuf_plan_copy_field(self._h, C.c_void_p(out.data_ptr())))
        return out

    def structure_factor(self, modes):
        """S~(n) for integer modes (K,3) within the cutoff sphere; complex128 numpy array."""
        import numpy as np
        ml = np.ascontiguousarray(np.asarray(modes, dtype=np.int32).reshape(-1, 3))
        out = np.empty(2 * ml.shape[0], dtype=np.float64)
        _check(lib().enuf_plan_structure_factor(self._h, ml.shape[0], ml.ctypes.data_as(C.POINTER(C.c_int)),
                                                out.ctypes.data_as(C.POINTER(C.c_double))))
        return out[0::2] + 1j * out[1::2]

    def close(self) -> None:
        if self._h:
            lib().enuf_plan_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def self_energy_static(q, alpha, out):
    """enuf_self_energy_static: E_self = (alpha / sqrt(pi)) sum q_i^2 of the CUDA tensor q (fp32 or fp64, contiguous)
    into the one-element fp64 CUDA tensor `out`, on torch's current stream, asynchronously.  Allocates nothing (the
    scratch is a static device array in the library): N <= SELF_STATIC_MAX_N, and calls that overlap on the GPU race."""
    import torch
    if not torch.cuda.is_available():
        raise EnufError(ECUDA, "no CUDA device available; this library has no CPU fallback")
    if not (isinstance(q, torch.Tensor) and q.is_cuda and q.is_contiguous() and q.dim() == 1
            and q.dtype in (torch.float32, torch.float64)):
        raise TypeError("q must be a contiguous 1-D CUDA tensor of float32 or float64")
    if not (isinstance(out, torch.Tensor) and out.is_cuda and out.dtype == torch.float64 and out.numel() == 1
            and out.device == q.device):
        raise TypeError("out must be a one-element float64 CUDA tensor on q's device")
    with torch.cuda.device(q.device):
        _check(lib().enuf_self_energy_static(C.c_void_p(q.data_ptr()), int(q.shape[0]),
                                             F32 if q.dtype == torch.float32 else F64, float(alpha),
                                             C.c_void_p(torch.cuda.current_stream().cuda_stream),
                                             C.c_void_p(out.data_ptr())))
    return out


def energy_forces(r, q, L, alpha, k_cut, M, sigma=2.0, m=6, **kw):
    """Convenience one-shot: create a plan, evaluate, destroy."""
    plan = Plan(q.shape[0], L, alpha, k_cut, M, sigma=sigma, m=m, dtype=r.dtype, **kw)
    try:
        return plan.energy_forces(r, q)
    finally:
        plan.close()
