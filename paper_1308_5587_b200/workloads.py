"""Seeded synthetic workloads shaped like the paper's LJ-liquid benchmark.

This module is the ONLY code shared by the CUDA path and the oracle: it makes
inputs and holds none of the method's arithmetic (no cell index, no distance,
no force, no integrator).  It imports neither `oracle/` nor the CUDA binding.

Recipe (the paper's own benchmark is PAPER.md:149,
"N=64000 particle Lennard-Jones fluid at packing fraction 0.20, r_cut=3.0,
k_B T = 1.2", whose script -- Algorithm 1, PAPER.md:75 -- is missing from the
text; these inputs stand in for it):

* n = ceil(N^(1/3)) simple-cubic sites at ((i+1/2) L/n - L/2); if n^3 > N a
  seeded-shuffle subset of N sites is kept;
* every coordinate jittered uniformly in +-jitter (0.05 sigma), wrapped into
  [-L/2, L/2);
* types by seeded shuffle (first floor(frac_A N) of the shuffled order are A);
* velocities Gaussian with sigma_v = sqrt(T*), mean subtracted, no rescale;
* all random numbers from a counter-based generator, splitmix64 of
  (seed, stream, index), so any language reproduces them;
* L, positions and velocities rounded ONCE to fp32; both sides read the same
  fp32 arrays.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)
_GOLDEN = np.uint64(0x9E3779B97F4A7C15)

STREAM_SITE, STREAM_JITTER, STREAM_TYPE, STREAM_VEL = 1, 2, 3, 4


def _mix64(z: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser (Steele, Lea, Flood 2014), vectorised on uint64."""
    z = z.astype(np.uint64, copy=True)
    with np.errstate(over="ignore"):
        z ^= z >> np.uint64(30)
        z *= np.uint64(0xBF58476D1CE4E5B9)
        z ^= z >> np.uint64(27)
        z *= np.uint64(0x94D049BB133111EB)
        z ^= z >> np.uint64(31)
    return z


def counter_u64(seed: int, stream: int, index: np.ndarray) -> np.ndarray:
    """64 random bits for each counter value: mix(mix(mix(seed)+stream*G)+index*G)."""
    index = np.asarray(index, dtype=np.uint64)
    with np.errstate(over="ignore"):
        s = _mix64(np.array([np.uint64(seed) + _GOLDEN], dtype=np.uint64))[0]
        s = _mix64(np.array([s + np.uint64(stream) * _GOLDEN], dtype=np.uint64))[0]
        return _mix64(s + (index + np.uint64(1)) * _GOLDEN)


def counter_uniform(seed: int, stream: int, index: np.ndarray) -> np.ndarray:
    """Uniform doubles in (0, 1): top 53 bits + 1/2 ulp, never 0 or 1."""
    u = counter_u64(seed, stream, index) >> np.uint64(11)
    return (u.astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def counter_normal(seed: int, stream: int, index: np.ndarray) -> np.ndarray:
    """Standard normals by Box-Muller from counters 2*index and 2*index+1."""
    index = np.asarray(index, dtype=np.uint64)
    u1 = counter_uniform(seed, stream, index * np.uint64(2))
    u2 = counter_uniform(seed, stream, index * np.uint64(2) + np.uint64(1))
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * math.pi * u2)


def seeded_permutation(seed: int, stream: int, n: int) -> np.ndarray:
    """Permutation of range(n): stable argsort of one 64-bit key per element."""
    keys = counter_u64(seed, stream, np.arange(n, dtype=np.uint64))
    return np.argsort(keys, kind="stable")


@dataclasses.dataclass(frozen=True)
class Workload:
    """One of BASELINE.json's configs.  Tables are row-major [ntypes][ntypes]."""
    name: str
    N: int
    rho: float
    T: float
    ntypes: int
    eps: tuple
    sigma: tuple
    rcut: tuple          # per type pair
    r_buff: float
    dt: float
    steps: int
    shift: int           # 0 = none, 1 = energy shift
    sort_period: int
    frac_A: float = 1.0
    jitter: float = 0.05
    seed: int = 0

    @property
    def L(self) -> float:
        """Cubic box edge, (N/rho)^(1/3), rounded once to fp32."""
        return float(np.float32((self.N / self.rho) ** (1.0 / 3.0)))

    @property
    def r_cut_max(self) -> float:
        return float(max(self.rcut))

    @property
    def r_max(self) -> float:
        return float(np.float32(np.float32(self.r_cut_max) + np.float32(self.r_buff)))


def _f32(x: float) -> float:
    return float(np.float32(x))


_WCA = _f32(2.0 ** (1.0 / 6.0))

CONFIGS = {
    # BASELINE.json configs[0..4]
    "lj_1k": Workload("lj_1k", 1_000, 0.382, 1.2, 1, (1.0,), (1.0,), (3.0,),
                      _f32(0.4), _f32(0.005), 10, 1, 0),
    "lj_64k": Workload("lj_64k", 64_000, 0.382, 1.2, 1, (1.0,), (1.0,), (3.0,),
                       _f32(0.4), _f32(0.005), 10_000, 1, 300),
    "lj_1m": Workload("lj_1m", 1_000_000, 0.382, 1.2, 1, (1.0,), (1.0,), (3.0,),
                      _f32(0.4), _f32(0.005), 5_000, 1, 300),
    "wca_256k": Workload("wca_256k", 256_000, 0.85, 1.0, 1, (1.0,), (1.0,), (_WCA,),
                         _f32(0.3), _f32(0.005), 10_000, 1, 300),
    "ka_1m": Workload("ka_1m", 1_048_576, 1.2, 1.0, 2,
                      (1.0, 1.5, 1.5, 0.5),
                      (1.0, _f32(0.8), _f32(0.8), _f32(0.88)),
                      (2.5, 2.0, 2.0, _f32(2.5 * 0.88)),
                      _f32(0.3), _f32(0.002), 5_000, 1, 300, frac_A=0.8),
}
CONFIG_ORDER = ["lj_1k", "lj_64k", "lj_1m", "wca_256k", "ka_1m"]


def scaled(w: Workload, N: int, **kw) -> Workload:
    """Same fluid at another particle count (parity cases below full size)."""
    return dataclasses.replace(w, name=f"{w.name}@{N}", N=N, **kw)


@dataclasses.dataclass
class State:
    L: float
    pos: np.ndarray      # float32 [N][3], in [-L/2, L/2)
    vel: np.ndarray      # float32 [N][3]
    type: np.ndarray     # int32 [N]
    image: np.ndarray    # int32 [N][3], zeros


def make_state(w: Workload, seed: int | None = None) -> State:
    seed = w.seed if seed is None else seed
    N, L = w.N, w.L
    n = int(math.ceil(N ** (1.0 / 3.0) - 1e-9))
    while n ** 3 < N:
        n += 1
    nsites = n ** 3
    if nsites > N:
        keep = np.sort(seeded_permutation(seed, STREAM_SITE, nsites)[:N])
    else:
        keep = np.arange(N)
    ix = keep % n
    iy = (keep // n) % n
    iz = keep // (n * n)
    site = np.stack([ix, iy, iz], axis=1).astype(np.float64)
    pos = (site + 0.5) * (L / n) - 0.5 * L
    k = np.arange(N * 3, dtype=np.uint64)
    pos += ((2.0 * counter_uniform(seed, STREAM_JITTER, k) - 1.0) * w.jitter).reshape(N, 3)
    pos -= L * np.floor((pos + 0.5 * L) / L)
    pos32 = pos.astype(np.float32)
    Lf = np.float32(L)
    half = np.float32(0.5) * Lf
    pos32 = np.where(pos32 >= half, pos32 - Lf, pos32)
    pos32 = np.where(pos32 < -half, pos32 + Lf, pos32).astype(np.float32)

    types = np.zeros(N, dtype=np.int32)
    if w.ntypes > 1:
        order = seeded_permutation(seed, STREAM_TYPE, N)
        nA = int(math.floor(w.frac_A * N))
        types[order[nA:]] = 1

    vel = counter_normal(seed, STREAM_VEL, k).reshape(N, 3) * math.sqrt(w.T)
    vel -= vel.mean(axis=0, keepdims=True)
    return State(L=L, pos=np.ascontiguousarray(pos32),
                 vel=np.ascontiguousarray(vel.astype(np.float32)),
                 type=types, image=np.zeros((N, 3), dtype=np.int32))


def uniform_random_state(N: int, L: float, T: float, seed: int, ntypes: int = 1) -> State:
    """Ideal-gas placement (uniform in the box); used by the pins that need an
    unstructured configuration (mean list length, faces/corners coverage)."""
    L = _f32(L)
    k = np.arange(N * 3, dtype=np.uint64)
    pos = (counter_uniform(seed, STREAM_JITTER, k).reshape(N, 3) - 0.5) * L
    pos32 = pos.astype(np.float32)
    Lf = np.float32(L)
    half = np.float32(0.5) * Lf
    pos32 = np.where(pos32 >= half, pos32 - Lf, pos32).astype(np.float32)
    vel = counter_normal(seed, STREAM_VEL, k).reshape(N, 3) * math.sqrt(T)
    vel -= vel.mean(axis=0, keepdims=True)
    types = (counter_u64(seed, STREAM_TYPE, np.arange(N, dtype=np.uint64)) % np.uint64(ntypes)).astype(np.int32)
    return State(L=L, pos=np.ascontiguousarray(pos32), vel=np.ascontiguousarray(vel.astype(np.float32)),
                 type=types, image=np.zeros((N, 3), dtype=np.int32))
