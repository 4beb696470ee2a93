"""Seeded input generators and literal plan parameters (see package docstring).

Config numbering follows BASELINE.json ``configs`` (1-based: cfg1 .. cfg5).
Plan parameters are literals taken from SURVEY.md section 8(d); the rule that produces
some of them (Eq. 31-32) is implemented separately by the
oracle and by the CUDA library, and the tests check both against these literals.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

_MASK = np.uint64(0xFFFFFFFFFFFFFFFF)
_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_C1 = np.uint64(0xBF58476D1CE4E5B9)
_C2 = np.uint64(0x94D049BB133111EB)


def splitmix64(seed: int, counter: np.ndarray) -> np.ndarray:
    """SplitMix64 output for ``state = seed + (counter + 1) * GOLDEN`` (uint64)."""
    with np.errstate(over="ignore"):
        c = np.asarray(counter, dtype=np.uint64)
        z = np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + (c + np.uint64(1)) * _GOLDEN
        z = (z ^ (z >> np.uint64(30))) * _C1
        z = (z ^ (z >> np.uint64(27))) * _C2
        z = z ^ (z >> np.uint64(31))
    return z


def uniform01(seed: int, counter: np.ndarray) -> np.ndarray:
    """fp64 uniform in [0, 1) from the 53 high bits."""
    return (splitmix64(seed, counter) >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)


def _gauss(seed: int, count: int) -> np.ndarray:
    """``count`` standard normals by Box-Muller (two uniforms per value)."""
    i = np.arange(count, dtype=np.uint64)
    u1 = uniform01(seed, 2 * i)
    u2 = uniform01(seed, 2 * i + 1)
    u1 = np.maximum(u1, 2.0 ** -53)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * math.pi * u2)


@dataclass
class Workload:
    name: str
    N: int
    L: float
    alpha: float
    k_cut: int
    M: int            # NFFT bandwidth per dimension
    sigma: float      # oversampling factor
    m: int            # window cut-off (support 2m+1 grid points)
    window: str       # "gaussian" | "kaiser_bessel"
    dtype: str        # "f64" | "f32"
    r: np.ndarray     # (N, 3) positions, dtype per config
    q: np.ndarray     # (N,) charges, dtype per config
    slater_lambda: float = 0.0   # 0 = point charges
    seed: int = 0
    meta: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        """Oversampled grid points per dimension, n = sigma * M."""
        return int(round(self.sigma * self.M))

    @property
    def np_dtype(self):
        return np.float64 if self.dtype == "f64" else np.float32


CONFIGS = ("cfg1", "cfg2", "cfg2_perfect", "cfg2_perfect_k16", "cfg3", "cfg4", "cfg5")


def _finish(name, r64, q64, dtype, **kw) -> Workload:
    dt = np.float64 if dtype == "f64" else np.float32
    r = np.ascontiguousarray(r64.astype(dt))
    q = np.ascontiguousarray(q64.astype(dt))
    return Workload(name=name, N=int(q.shape[0]), r=r, q=q, dtype=dtype, **kw)


def _cfg1():
    N, L, seed = 1000, 10.0, 1001
    r = uniform01(seed, np.arange(3 * N)).reshape(N, 3) * L
    q = np.where(np.arange(N) % 2 == 0, 1.0, -1.0)
    return _finish("cfg1", r, q, "f64", L=L, alpha=2.0 * math.pi / L, k_cut=8, M=16,
                   sigma=2.0, m=4, window="gaussian", seed=seed)


def _rock_salt(cells: int, a: float):
    """Rock salt = simple cubic lattice of spacing a/2 with charge (-1)^(i+j+k)."""
    g = 2 * cells
    idx = np.arange(g)
    i, j, k = np.meshgrid(idx, idx, idx, indexing="ij")
    r = np.stack([i, j, k], axis=-1).reshape(-1, 3).astype(np.float64) * (a / 2.0)
    q = np.where((i + j + k).reshape(-1) % 2 == 0, 1.0, -1.0)
    return r, q


def _cfg2(perfect: bool, k_cut: int, name: str):
    cells, a, seed = 8, 1.0, 2002
    L = cells * a
    r, q = _rock_salt(cells, a)
    if not perfect:
        r = r + 0.05 * a * _gauss(seed, r.size).reshape(r.shape)
        r = r - np.floor(r / L) * L
    # BASELINE's "alpha=3.5" is read as 3.5*pi/L.
    return _finish(name, r, q, "f64", L=L, alpha=3.5 * math.pi / L, k_cut=k_cut, M=32,
                   sigma=2.0, m=6, window="kaiser_bessel", seed=seed,
                   meta={"r0": a / 2.0, "perfect": perfect})


def _cfg3():
    N, L, seed = 24000, 20.0, 3003
    r = uniform01(seed, np.arange(3 * N)).reshape(N, 3) * L
    q = np.zeros(N)
    q[:2400] = 1.0
    q[2400:4800] = -1.0
    return _finish("cfg3", r, q, "f32", L=L, alpha=0.9, k_cut=18, M=64, sigma=2.0, m=4,
                   window="gaussian", slater_lambda=0.25, seed=seed, meta={"delta": 1e-4})


def _cfg4():
    n_mol, L, seed, radius = 12500, 100.0, 4004, 2.0
    cat = 0.8 * np.array([0.4, 0.3, 0.15, 0.1, 0.05])
    ani = -0.8 * np.array([0.5, 0.25, 0.25])
    sites = np.concatenate([np.full(n_mol, 5), np.full(n_mol, 3)])
    first = np.concatenate([[0], np.cumsum(sites)])
    N = int(first[-1])
    n_molecules = 2 * n_mol
    centres = uniform01(seed, np.arange(3 * n_molecules)).reshape(n_molecules, 3) * L
    # site offsets: uniform in a ball of radius 2 (direction from a Gaussian triple,
    # radius from U^(1/3)); counters continue after the centres.
    base = 3 * n_molecules
    gs = _gauss(seed + 1, 3 * N).reshape(N, 3)
    gs /= np.linalg.norm(gs, axis=1, keepdims=True)
    rad = radius * np.cbrt(uniform01(seed, base + np.arange(N)))
    mol_of_site = np.repeat(np.arange(n_molecules), sites)
    r = centres[mol_of_site] + gs * rad[:, None]
    r = r - np.floor(r / L) * L
    q = np.concatenate([np.tile(cat, n_mol), np.tile(ani, n_mol)])
    return _finish("cfg4", r, q, "f32", L=L, alpha=0.3, k_cut=33, M=128, sigma=2.0, m=6,
                   window="kaiser_bessel", seed=seed, meta={"delta": 1e-5})


def _cfg5(N: int = 1_000_000, sigma: float = 2.0, name: str = "cfg5"):
    L, seed = 215.0, 5005
    r = uniform01(seed, np.arange(3 * N)).reshape(N, 3) * L
    q = np.where(np.arange(N) % 2 == 0, 1.0, -1.0)
    r_c, delta = 10.0, 1e-4
    alpha = math.sqrt(-math.log(delta)) / r_c          # 0.30348542587702925
    return _finish(name, r, q, "f32", L=L, alpha=alpha, k_cut=64, M=128, sigma=sigma, m=6,
                   window="kaiser_bessel", seed=seed,
                   meta={"delta": delta, "r_c": r_c, "step_displacement": 0.05})


def make_workload(name: str) -> Workload:
    if name == "cfg1":
        return _cfg1()
    if name == "cfg2":
        return _cfg2(False, 12, name)
    if name == "cfg2_perfect":
        return _cfg2(True, 12, name)
    if name == "cfg2_perfect_k16":
        return _cfg2(True, 16, name)
    if name == "cfg3":
        return _cfg3()
    if name == "cfg4":
        return _cfg4()
    if name == "cfg5":
        return _cfg5()
    if name == "cfg5_sigma15":      # config 5 on the 192^3 grid of sigma_s = 1.5; same inputs
        return _cfg5(sigma=1.5, name=name)
    raise KeyError(name)


def displaced_positions(r: np.ndarray, L: float, seed: int, step: int, amplitude: float) -> np.ndarray:
    """One config-5 step: r <- wrap(r + amplitude*(2U-1)), U = hash(seed, step, j, d).

    The displacement is formed in fp64, rounded to r's dtype, added with one add in
    r's dtype and wrapped into [0, L) in that dtype (integer-exact hash on both sides).
    """
    N = r.shape[0]
    ctr = np.uint64(step) * np.uint64(3 * N) + np.arange(3 * N, dtype=np.uint64)
    u = uniform01(seed ^ 0x5DEECE66D, ctr).reshape(N, 3)
    d = (amplitude * (2.0 * u - 1.0)).astype(r.dtype)
    out = r + d
    Lt = r.dtype.type(L)
    out = np.where(out < 0, out + Lt, out)
    out = np.where(out >= Lt, out - Lt, out)
    return np.ascontiguousarray(out.astype(r.dtype))


def random_neutral_gas(N: int, L: float, seed: int, dtype=np.float64):
    """Small neutral +-1 gas for brute-force and edge-case tests."""
    r = uniform01(seed, np.arange(3 * N)).reshape(N, 3) * L
    q = np.where(np.arange(N) % 2 == 0, 1.0, -1.0)
    return np.ascontiguousarray(r.astype(dtype)), np.ascontiguousarray(q.astype(dtype))
