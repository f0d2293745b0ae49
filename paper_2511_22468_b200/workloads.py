"""Seeded synthetic workloads shaped like the paper's: Plummer-sphere progenitors
on Milky-Way orbits (section 2.1 "tidal disruption of a Plummer sphere in
a realistic Milky Way potential"; L43 Fig. 2 step 3 "sampled from a Plummer
sphere in equilibrium"; L47 "shifted in phase space").

This module is the ONE piece both the oracle tests and the CUDA path use.  It
holds input generation only -- none of the method's arithmetic (no force, no
potential, no integrator) -- is pure numpy fp64 on the host, and imports neither
``oracle`` nor the CUDA binding.  The configuration table restates
BASELINE.json ``configs[0..4]``; the recipe is DESIGN.md section "Input recipe".
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional, Tuple

import numpy as np

G_KPC_MSUN_MYR = 4.4985e-12        # kpc^3 Msun^-1 Myr^-2 (BASELINE.json configs[1])
NFW_MW = (1.0e12, 16.0)            # M_s [Msun], r_s [kpc]
MN_MW = (6.8e10, 3.0, 0.28)        # M [Msun], a [kpc], b [kpc]


@dataclass(frozen=True)
class Config:
    name: str
    n: int
    G: float
    M: float                       # progenitor total mass
    a: float                       # Plummer scale radius
    eps: float                     # softening length
    dt: float
    nsteps: int
    centre: Tuple[float, float, float] = (0.0, 0.0, 0.0)
    velocity: Tuple[float, float, float] = (0.0, 0.0, 0.0)
    nfw: Optional[Tuple[float, float]] = None
    mn: Optional[Tuple[float, float, float]] = None
    precisions: Tuple[str, ...] = ("f32",)
    seed: int = 1000
    note: str = ""


_GD1 = dict(centre=(-10.0, -4.0, 6.0), velocity=(0.12, -0.18, -0.08))

# BASELINE.json configs[0..4]; seeds = 1000 + index.  Configs 3-4 take
# config 2's orbit start (reading R19).
CONFIGS = (
    Config("cfg0_plummer_isolated_n1024", 1024, 1.0, 1.0, 1.0, 0.01, 1e-3, 10,
           precisions=("f64", "f32"), seed=1000,
           note="N-body units G=M=a=1, no external potential"),
    Config("cfg1_progenitor_mw_n16384", 16384, G_KPC_MSUN_MYR, 1.0e4, 0.010, 0.001, 0.5, 1000,
           centre=(12.4, 0.0, 1.5), velocity=(0.0, 0.21, 0.05), nfw=NFW_MW, mn=MN_MW, seed=1001),
    Config("cfg2_gd1_stream_n65536", 65536, G_KPC_MSUN_MYR, 5.0e4, 0.015, 0.001, 1.0, 3000,
           nfw=NFW_MW, mn=MN_MW, seed=1002, **_GD1),
    Config("cfg3_disruption_n262144", 262144, G_KPC_MSUN_MYR, 1.0e5, 0.020, 0.0005, 0.5, 200,
           nfw=NFW_MW, mn=MN_MW, precisions=("f32", "f64"), seed=1003, **_GD1),
    Config("cfg4_disruption_n1048576", 1048576, G_KPC_MSUN_MYR, 1.0e6, 0.050, 0.0005, 0.5, 20,
           nfw=NFW_MW, mn=MN_MW, seed=1004, **_GD1),
)

TARGET_SUBSET_SEED = 99
TARGET_SUBSET_SIZE = 4096


def _isotropic(rng: np.random.Generator, n: int) -> np.ndarray:
    cos_t = rng.uniform(-1.0, 1.0, n)
    phi = rng.uniform(0.0, 2.0 * np.pi, n)
    sin_t = np.sqrt(np.maximum(0.0, 1.0 - cos_t * cos_t))
    return np.stack([sin_t * np.cos(phi), sin_t * np.sin(phi), cos_t], axis=1)


def plummer_sphere(n: int, G: float, M: float, a: float, seed: int):
    """Equal-mass equilibrium Plummer sphere, fp64, recentred on its centre of mass.

    Recipe (BASELINE.json configs[0]; reading R13): radius by inverse CDF
    r = a / sqrt(u^(-2/3) - 1), u in (0, 1) open, no truncation; isotropic direction;
    speed v = q * v_esc(r), v_esc = sqrt(2 G M / a) (1 + r^2/a^2)^(-1/4), q by von Neumann
    rejection on g(q) = q^2 (1 - q^2)^(7/2) under the box [0,1) x [0,0.1); isotropic
    velocity direction; masses M/n.  PRNG: numpy Generator(PCG64(seed)).
    Returns (posm [n,4], vel [n,3]).
    """
    rng = np.random.Generator(np.random.PCG64(seed))
    u = rng.uniform(0.0, 1.0, n)
    u = np.where(u <= 0.0, np.nextafter(0.0, 1.0), u)
    r = a / np.sqrt(u ** (-2.0 / 3.0) - 1.0)
    pos = r[:, None] * _isotropic(rng, n)
    q = np.empty(n)
    todo = np.arange(n)
    while todo.size:
        qq = rng.uniform(0.0, 1.0, todo.size)
        yy = rng.uniform(0.0, 0.1, todo.size)
        ok = yy < qq * qq * (1.0 - qq * qq) ** 3.5
        q[todo[ok]] = qq[ok]
        todo = todo[~ok]
    v_esc = np.sqrt(2.0 * G * M / a) * (1.0 + (r / a) ** 2) ** (-0.25)
    vel = (q * v_esc)[:, None] * _isotropic(rng, n)
    m = np.full(n, M / n)
    pos -= np.mean(pos, axis=0)          # equal masses: mass-weighted mean == mean
    vel -= np.mean(vel, axis=0)
    posm = np.concatenate([pos, m[:, None]], axis=1)
    return np.ascontiguousarray(posm), np.ascontiguousarray(vel)


def make_state(cfg: Config, n: Optional[int] = None, seed: Optional[int] = None):
    """fp64 initial state of a config: Plummer sphere shifted to the orbit start.

    ``n`` overrides the particle count (same shape, smaller case).  fp32 runs cast
    once (round-to-nearest) AFTER the shift, with ``to_f32``.
    """
    posm, vel = plummer_sphere(n or cfg.n, cfg.G, cfg.M, cfg.a, cfg.seed if seed is None else seed)
    posm[:, :3] += np.asarray(cfg.centre, dtype=np.float64)
    vel += np.asarray(cfg.velocity, dtype=np.float64)
    return posm, vel


def to_f32(a: np.ndarray) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float32)


def vel4(vel: np.ndarray, dtype) -> np.ndarray:
    """[n,3] -> [n,4] record with zero padding lane (device layout)."""
    out = np.zeros((vel.shape[0], 4), dtype=dtype)
    out[:, :3] = vel
    return out


def target_subset(n: int, size: int = TARGET_SUBSET_SIZE, seed: int = TARGET_SUBSET_SEED) -> np.ndarray:
    """Seeded, sorted, duplicate-free sample of target indices (config 4's 4,096-target check)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    size = min(size, n)
    return np.sort(rng.choice(n, size=size, replace=False)).astype(np.int64)


def random_cloud(n: int, seed: int, scale: float = 1.0, centre=(0.0, 0.0, 0.0), unequal_mass: bool = True):
    """Plain Gaussian cloud with unequal masses: edge-case / ragged-size parity input."""
    rng = np.random.Generator(np.random.PCG64(seed))
    pos = rng.normal(0.0, scale, (n, 3)) + np.asarray(centre, dtype=np.float64)
    m = rng.uniform(0.5, 1.5, n) if unequal_mass else np.ones(n)
    vel = rng.normal(0.0, 0.1, (n, 3))
    return np.ascontiguousarray(np.concatenate([pos, m[:, None]], axis=1)), np.ascontiguousarray(vel)
