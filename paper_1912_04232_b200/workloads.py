"""Seeded synthetic inputs for the five BASELINE.json configs.

This module is the ONE piece shared by the CUDA path, the oracle and the tests:
it draws random numbers and lays particles out, and holds none of the method's
arithmetic (no displacement, no cell index, no energy, no integrator).  It
imports neither ``oracle/`` nor the CUDA binding.

The paper's benchmark is "Lennard-Jones particles ... a ubiquitous performance
benchmark" (§3.1) with no dataset behind it, and the bidisperse
soft-disk packing of PAPER.md:L134 §4.2 / L293-L305 App. A.  The configs below
stand in for those workloads; the recipe is restated in DESIGN.md §4.

Every array is generated in fp64 from ``numpy.random.default_rng(SEED0 + index)``
and cast to fp32 ONCE; the fp32 arrays are the single input to both sides.
Layout: ``pos`` float32[N,4] = (x, y, z, w) with w = particle diameter
(soft sphere) or 1.0 (LJ, unused); ``vel`` float32[N,4] = (vx, vy, vz, 0).
In 2-D z = 0 and vz = 0.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

SEED0 = 19120423          # arXiv id 1912.04232 (+ config index)
RHO_LJ = 0.8442           # LJ number density of configs 0, 2, 3, 4

KIND_LJ = 0
KIND_SOFT = 1
KIND_MORSE = 2
KIND_BUCKINGHAM = 3
KIND_LJ_SPECIES = 4
KIND_BKS = 5


@dataclasses.dataclass(frozen=True)
class Workload:
    """One BASELINE.json config: parameters + the fp32 initial state."""
    index: int
    name: str
    dim: int
    n: int
    box: np.ndarray          # float32[3]; box[2] = 1 in 2-D (ignored)
    kind: int                # KIND_LJ | KIND_SOFT
    epsilon: float
    sigma: float
    r_cut: float             # list radius is r_cut + skin; LJ truncation radius
    skin: float
    capacity: int
    shift: int               # 1: u(r) - u(r_cut)
    dt: float
    mass: float
    temperature: float
    steps: int
    resort: int
    pos: np.ndarray          # float32[N,4]
    vel: np.ndarray          # float32[N,4]
    alpha: float = 0.0       # Morse inverse width (KIND_MORSE: sigma = r0, epsilon = D)

    @property
    def list_radius(self) -> float:
        return float(np.float32(self.r_cut) + np.float32(self.skin))


def fcc_sites(m: int, a: float) -> np.ndarray:
    """The 4*m^3 sites of an FCC lattice with cubic cell edge ``a`` (fp64)."""
    basis = np.array([[0.0, 0.0, 0.0], [0.5, 0.5, 0.0],
                      [0.5, 0.0, 0.5], [0.0, 0.5, 0.5]])
    g = np.arange(m, dtype=np.float64)
    cells = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 1, 3)
    return ((cells + basis[None, :, :]) * a).reshape(-1, 3)


def into_box_f32(x64: np.ndarray, box32: np.ndarray) -> np.ndarray:
    """Place fp64 coordinates into [0, L) and cast to fp32 so that the fp32
    value still satisfies 0 <= x < L (input conditioning only)."""
    L = box32.astype(np.float64)
    x = np.mod(x64, L[None, : x64.shape[1]])
    x32 = x.astype(np.float32)
    Lc = box32[None, : x64.shape[1]]
    x32 = np.where(x32 >= Lc, np.float32(0.0), x32)
    x32 = np.where(x32 < 0, np.float32(0.0), x32)
    return x32.astype(np.float32)


def maxwell_boltzmann(rng, n: int, dim: int, temperature: float, mass: float) -> np.ndarray:
    """N(0, T/m) per component, zero net momentum, rescaled so that
    sum(m v^2) / (dim (N-1)) = T exactly (fp64)."""
    if temperature == 0.0:
        return np.zeros((n, dim))
    v = rng.normal(0.0, math.sqrt(temperature / mass), size=(n, dim))
    v -= v.mean(axis=0, keepdims=True)
    t_now = mass * (v * v).sum() / (dim * (n - 1))
    v *= math.sqrt(temperature / t_now)
    return v


def _pack(x32: np.ndarray, w: np.ndarray | float) -> np.ndarray:
    n, d = x32.shape
    out = np.zeros((n, 4), dtype=np.float32)
    out[:, :d] = x32
    out[:, 3] = w
    return out


def lj_fcc(index: int, m: int, *, temperature: float = 1.0, skin: float = 0.3,
           steps: int = 100, resort: int = 1, jitter: float = 0.05,
           seed: int | None = None, name: str | None = None, rho: float = RHO_LJ) -> Workload:
    """3-D LJ fluid on a jittered FCC lattice at rho = 0.8442 (configs 0,2,3,4; other densities: tests)."""
    n = 4 * m ** 3
    L64 = (n / rho) ** (1.0 / 3.0)
    box = np.array([L64, L64, L64], dtype=np.float32)
    rng = np.random.default_rng(SEED0 + index if seed is None else seed)
    sites = fcc_sites(m, float(box[0]) / m)
    x = sites + rng.normal(0.0, jitter, size=sites.shape) if jitter > 0 else sites
    pos = _pack(into_box_f32(x, box), 1.0)
    v = maxwell_boltzmann(rng, n, 3, temperature, 1.0)
    vel = _pack(v.astype(np.float32), 0.0)
    return Workload(index=index, name=name or f"lj3d_n{n}", dim=3, n=n, box=box,
                    kind=KIND_LJ, epsilon=1.0, sigma=1.0, r_cut=2.5, skin=skin,
                    capacity=128, shift=1, dt=0.005, mass=1.0,
                    temperature=temperature, steps=steps, resort=resort,
                    pos=pos, vel=vel)


def soft_disks(index: int = 1, n: int = 16384, *, phi: float = 0.90,
               d_small: float = 1.0, d_large: float = 1.4, steps: int = 1000,
               seed: int | None = None) -> Workload:
    """2-D 50:50 bidisperse harmonic soft disks at packing fraction phi
    (config 1; box from PAPER.md:L293-L295, species layout L297)."""
    n2 = n // 2
    area = n2 * math.pi * (d_small ** 2 + d_large ** 2) / 4.0
    L64 = math.sqrt(area / phi)
    box = np.array([L64, L64, 1.0], dtype=np.float32)
    rng = np.random.default_rng(SEED0 + index if seed is None else seed)
    x = rng.uniform(0.0, 1.0, size=(n, 2)) * float(box[0])
    diam = np.concatenate([np.full(n2, d_small), np.full(n - n2, d_large)])
    pos = _pack(into_box_f32(x, box), diam.astype(np.float32))
    vel = np.zeros((n, 4), dtype=np.float32)
    return Workload(index=index, name=f"soft2d_n{n}", dim=2, n=n, box=box,
                    kind=KIND_SOFT, epsilon=1.0, sigma=1.0, r_cut=d_large,
                    skin=0.1, capacity=32, shift=0, dt=0.01, mass=1.0,
                    temperature=0.0, steps=steps, resort=1, pos=pos, vel=vel)


def config(index: int, replica: int = 0) -> Workload:
    """BASELINE.json ``configs[index]``; ``replica`` > 0 draws an independent sample of the
    same workload (seed + 1000 * replica) for multi-GPU replica runs."""
    seed = SEED0 + index + 1000 * replica
    if index == 0:
        return lj_fcc(0, 6, steps=100, seed=seed)
    if index == 1:
        return soft_disks(1, 16384, steps=1000, seed=seed)
    if index == 2:
        return lj_fcc(2, 20, steps=1000, seed=seed)
    if index == 3:
        return lj_fcc(3, 40, steps=1000, seed=seed)
    if index == 4:
        return lj_fcc(4, 64, temperature=2.0, skin=0.2, steps=500, seed=seed)
    raise ValueError(f"no config {index}")


def random_box(seed: int, n: int, dim: int, box, *, diam=(1.0, 1.0)) -> tuple[np.ndarray, np.ndarray]:
    """Uniform random particles in an arbitrary box (test inputs)."""
    rng = np.random.default_rng(seed)
    box32 = np.array(list(box) + [1.0] * (3 - len(box)), dtype=np.float32)
    x = rng.uniform(0.0, 1.0, size=(n, dim)) * box32[None, :dim].astype(np.float64)
    w = np.where(np.arange(n) < n // 2, diam[0], diam[1]).astype(np.float32)
    return _pack(into_box_f32(x, box32), w), box32
