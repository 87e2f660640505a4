"""Seeded synthetic workloads (BASELINE.json configs 0-4; SURVEY.md §8d recipe).

This module serves BOTH the CUDA path and the oracle.  It holds no arithmetic of the
method (no kernels, no forces, no cell keys): it only draws particle positions,
velocities, internal energies and masses from the stated distributions with a
counter-based generator (numpy Philox keyed by (seed, stream)), in FP64, and rounds
once to the FP32 arrays both sides read.

The paper measures on its own galaxy-collision model whose parameters are not
printed ("quasi-isothermal model ... King model", L211-213); these
generators stand in for it.

Layout of what is returned (the boundary's layout, include/sph_b200.h):
  posm[N,4] float32 = (x, y, z, m)      vele[N,4] float32 = (vx, vy, vz, e)
gas particles first [0, N_g), halo particles [N_g, N).  Within each species the
order is [galaxy A, galaxy B].
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

__all__ = ["Workload", "CONFIGS", "make_workload", "lattice", "subset_indices"]


@dataclass
class Workload:
    name: str
    posm: np.ndarray          # [N,4] float32
    vele: np.ndarray          # [N,4] float32
    n_gas: int
    n_halo: int
    h: float
    delta: float
    G: float
    dt: float
    steps: int
    seed: int
    gamma: float = 5.0 / 3.0
    alpha: float = 0.5
    beta: float = 1.0
    eta: float = 0.1
    meta: dict = field(default_factory=dict)

    def __post_init__(self):
        # the boundary carries every parameter as FP32 (sph_params, dt): round them once here so
        # the oracle (FP64) and the CUDA path see bit-identical parameter values
        for k in ("h", "delta", "G", "dt", "gamma", "alpha", "beta", "eta"):
            object.__setattr__(self, k, float(np.float32(getattr(self, k))))

    def __setattr__(self, k, v):
        if k in ("h", "delta", "G", "dt", "gamma", "alpha", "beta", "eta"):
            v = float(np.float32(v))
        object.__setattr__(self, k, v)

    @property
    def n_total(self) -> int:
        return self.n_gas + self.n_halo


def _rng(seed: int, stream: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(key=[int(seed), int(stream)]))


def _invert_cdf(u: np.ndarray, mass_fn, x_max: float) -> np.ndarray:
    """Solve mass_fn(x)/mass_fn(x_max) = u for x in [0, x_max] by 64 bisection steps (FP64)."""
    target = u * mass_fn(np.float64(x_max))
    lo = np.zeros_like(u)
    hi = np.full_like(u, x_max)
    for _ in range(64):
        mid = 0.5 * (lo + hi)
        below = mass_fn(mid) < target
        lo = np.where(below, mid, lo)
        hi = np.where(below, hi, mid)
    return 0.5 * (lo + hi)


def _king_mass(x):
    # enclosed mass of rho ∝ (1+x^2)^(-3/2):  asinh(x) - x/sqrt(1+x^2)
    return np.arcsinh(x) - x / np.sqrt(1.0 + x * x)


def _qiso_mass(x):
    # enclosed mass of rho ∝ 1/(1+x^2):  x - atan(x)
    return x - np.arctan(x)


def _sphere(rng: np.random.Generator, n: int, mass_fn, core: float, r_trunc: float) -> np.ndarray:
    u = rng.random(n)
    r = core * _invert_cdf(u, mass_fn, r_trunc / core)
    cos_t = 2.0 * rng.random(n) - 1.0
    phi = 2.0 * np.pi * rng.random(n)
    sin_t = np.sqrt(np.maximum(0.0, 1.0 - cos_t * cos_t))
    return np.stack([r * sin_t * np.cos(phi), r * sin_t * np.sin(phi), r * cos_t], axis=1)


def _galaxy(seed, stream0, n_gas, n_halo, centre, bulk, gas_core, halo_core):
    """One galaxy: gas sphere (King-like, r<=10) inside a halo (quasi-isothermal, r<=20)."""
    centre = np.asarray(centre, dtype=np.float64)
    bulk = np.asarray(bulk, dtype=np.float64)
    g_pos = _sphere(_rng(seed, stream0 + 0), n_gas, _king_mass, gas_core, 10.0) + centre
    h_pos = _sphere(_rng(seed, stream0 + 1), n_halo, _qiso_mass, halo_core, 20.0) + centre
    g_vel = 0.3 * _rng(seed, stream0 + 2).standard_normal((n_gas, 3)) + bulk
    h_vel = 0.5 * _rng(seed, stream0 + 3).standard_normal((n_halo, 3)) + bulk
    g_e = 0.5 + 0.5 * _rng(seed, stream0 + 4).random(n_gas)
    return g_pos, h_pos, g_vel, h_vel, g_e


def _assemble(gas_pos, halo_pos, gas_vel, halo_vel, gas_e, mass):
    n_gas, n_halo = len(gas_pos), len(halo_pos)
    n = n_gas + n_halo
    posm = np.empty((n, 4), dtype=np.float32)
    vele = np.zeros((n, 4), dtype=np.float32)
    posm[:n_gas, :3] = gas_pos
    posm[n_gas:, :3] = halo_pos
    posm[:, 3] = np.float32(mass)
    vele[:n_gas, :3] = gas_vel
    vele[n_gas:, :3] = halo_vel
    vele[:n_gas, 3] = gas_e
    return posm, vele


def _single_galaxy(name, n_gas, n_halo, h, delta, dt, steps, seed):
    g_pos, h_pos, g_vel, h_vel, g_e = _galaxy(seed, 0, n_gas, n_halo, (0, 0, 0), (0, 0, 0), 1.0, 2.0)
    posm, vele = _assemble(g_pos, h_pos, g_vel, h_vel, g_e, 1.0 / (n_gas + n_halo))
    return Workload(name, posm, vele, n_gas, n_halo, h, delta, 1.0, dt, steps, seed)


def _collision(name, n_gas, n_halo, h, delta, dt, steps, seed, gas_core=1.0, halo_core=2.0):
    # centres (+8,+1,0) / (-8,-1,0), bulk velocities (-0.5,0,0) / (+0.5,0,0)
    a = _galaxy(seed, 0, n_gas // 2, n_halo // 2, (8, 1, 0), (-0.5, 0, 0), gas_core, halo_core)
    b = _galaxy(seed, 16, n_gas - n_gas // 2, n_halo - n_halo // 2, (-8, -1, 0), (0.5, 0, 0), gas_core, halo_core)
    cat = [np.concatenate([a[i], b[i]], axis=0) for i in range(5)]
    posm, vele = _assemble(cat[0], cat[1], cat[2], cat[3], cat[4], 1.0 / (n_gas + n_halo))
    return Workload(name, posm, vele, n_gas, n_halo, h, delta, 1.0, dt, steps, seed)


def _clumps(name, n_gas, h, seed):
    n_u = n_gas // 2
    n_c = n_gas - n_u
    uni = 2.0 * _rng(seed, 0).random((n_u, 3)) - 1.0
    centres = 2.0 * _rng(seed, 1).random((64, 3)) - 1.0
    which = _rng(seed, 2).integers(0, 64, size=n_c)
    clump = centres[which] + 0.02 * _rng(seed, 3).standard_normal((n_c, 3))
    pos = np.concatenate([uni, clump], axis=0)
    vel = 0.1 * _rng(seed, 4).standard_normal((n_gas, 3))
    e = 0.5 + 0.5 * _rng(seed, 5).random(n_gas)
    posm, vele = _assemble(pos, np.zeros((0, 3)), vel, np.zeros((0, 3)), e, 1.0 / n_gas)
    # no gravity in this config (BASELINE.json config 4): G = 0, delta kept positive
    return Workload(name, posm, vele, n_gas, 0, h, 0.001, 0.0, 1e-4, 1, seed)


CONFIGS = {
    0: dict(kind="single", n_gas=4096, n_halo=4096, h=0.2, delta=0.01, dt=1e-3, steps=1, seed=1),
    1: dict(kind="collision", n_gas=2 ** 16, n_halo=2 ** 16, h=0.1, delta=0.005, dt=5e-4, steps=10, seed=2),
    2: dict(kind="collision", n_gas=2 ** 19, n_halo=2 ** 19, h=0.05, delta=0.002, dt=2.5e-4, steps=10, seed=3),
    3: dict(kind="collision", n_gas=2 ** 21, n_halo=2 ** 21, h=0.02, delta=0.001, dt=1e-4, steps=5, seed=4,
            gas_core=0.2, halo_core=0.5),
    4: dict(kind="clumps", n_gas=2 ** 24, h=0.004, seed=5),
    # not a BASELINE.json config: SURVEY §8(f) NEXT-3, the collisionless mode (N_g = 0; SP, DC, HFC skipped,
    # PAPER.md L150) at N = 2^22, inside the paper's range of N (L213); same halo profile and orbits as config 2
    5: dict(kind="collision", n_gas=0, n_halo=2 ** 22, h=0.05, delta=0.001, dt=1e-4, steps=5, seed=6),
    # the same at N = 2^23, the top of the paper's range (L213)
    6: dict(kind="collision", n_gas=0, n_halo=2 ** 23, h=0.05, delta=0.001, dt=1e-4, steps=2, seed=7),
}


def make_workload(config: int, scale: float = 1.0) -> Workload:
    """Build BASELINE.json config `config`.  `scale` < 1 shrinks the particle counts
    (same distributions, same h) for quick tests; scale = 1 is the stated size."""
    c = dict(CONFIGS[config])
    kind = c.pop("kind")
    name = f"config{config}" + ("" if scale == 1.0 else f"@{scale:g}")
    if kind == "clumps":
        return _clumps(name, max(2, int(c["n_gas"] * scale)), c["h"], c["seed"])
    c["n_gas"] = max(2, int(c["n_gas"] * scale)) if c["n_gas"] else 0
    c["n_halo"] = max(2, int(c["n_halo"] * scale)) if c["n_halo"] else 0
    if kind == "single":
        return _single_galaxy(name, **c)
    return _collision(name, **c)


def lattice(n_side: int, spacing: float, rho0: float = 1.0, e: float = 1.0) -> Workload:
    """Uniform cubic lattice of gas, m = rho0 * spacing^3 (pin P3 input; no halo)."""
    ax = (np.arange(n_side, dtype=np.float64) - 0.5 * (n_side - 1)) * spacing
    x, y, z = np.meshgrid(ax, ax, ax, indexing="ij")
    pos = np.stack([x.ravel(), y.ravel(), z.ravel()], axis=1)
    n = len(pos)
    posm, vele = _assemble(pos, np.zeros((0, 3)), np.zeros((n, 3)), np.zeros((0, 3)), np.full(n, e),
                           rho0 * spacing ** 3)
    return Workload(f"lattice{n_side}", posm, vele, n, 0, spacing, 0.01, 0.0, 1e-3, 1, 0)


def subset_indices(n_gas: int, n_halo: int, seed: int, n_each: int = 2048):
    """Seeded subset for the large-N protocol: n_each gas + n_each halo
    indices without replacement (global particle numbering), ascending."""
    g = np.sort(_rng(seed, 1000).choice(n_gas, size=min(n_each, n_gas), replace=False)) if n_gas else np.zeros(0, int)
    hh = np.sort(_rng(seed, 1001).choice(n_halo, size=min(n_each, n_halo), replace=False)) + n_gas if n_halo \
        else np.zeros(0, int)
    return g.astype(np.int64), hh.astype(np.int64)
