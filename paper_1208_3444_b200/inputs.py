"""Seeded synthetic input generators for the five BASELINE.json configs.

This module serves BOTH the CUDA path and the CPU oracle (tests hand the same
float32 bytes to each side).  It holds none of the method's arithmetic: no
force, no integrator, no Friedmann equation -- only particle placement, masses
and the per-config constants.
It imports neither `oracle` nor the CUDA binding.

The paper's own workload (glass + Zel'dovich + Eisenstein-Hu initial conditions
read from a data file) is not available; config 2 takes
its shape (32^3 particles in a unit box standing for 100 Mpc, z = 50 start,
near-uniform, zero velocities) and stands in for it.

Random numbers: numpy `Generator(PCG64(seed))`.  Arrays are produced in float64
and rounded once to float32; the float32 arrays are the inputs of record.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

__all__ = ["Config", "CONFIGS", "make_config", "sample_targets", "pack_pos_mass"]


@dataclass(frozen=True)
class Cosmology:
    """The five numbers of eq. (2), PAPER.md:33 (G10: caller passes all five)."""
    H0: float
    Om_R: float = 0.0
    Om_M: float = 0.0
    Om_K: float = 0.0
    Om_L: float = 0.0


@dataclass(frozen=True)
class Config:
    index: int                  # 1..5 as in BASELINE.json `configs`
    name: str
    n: int
    seed: int
    eps: float                  # softening length (decimal); eps2 below is what both sides use
    G: float
    steps: int                  # trajectory steps of the config (0 = force only)
    parity_steps: int           # steps compared particle by particle (north_star: 10)
    tau: float                  # constant step in cosmic time t (G9)
    cosmo: Cosmology | None     # None = static background a=1, H=0 (config 3)
    a_start: float              # scale factor at step 0
    n_tracers: int = 0
    tracer_stride: int = 0
    oracle_targets: int = 0     # 0 = all targets; else number of sampled targets
    extra: dict = field(default_factory=dict)

    @property
    def eps2(self) -> np.float32:
        """eps^2 as the float32 value passed through the ABI (G6)."""
        return np.float32(np.float32(self.eps) * np.float32(self.eps))


_H0_EDS = math.sqrt(8.0 * math.pi / 3.0)            # G13: box holds the critical density, G=1
_G_LCDM = 3.0 * 0.3 * 70.0 ** 2 / (8.0 * math.pi)   # G13: rho_bar = Om_M 3 H0^2 / (8 pi G) = 1

CONFIGS = {
    1: Config(1, "uniform-4096-EdS", 4096, 0, 0.01, 1.0, 10, 10, 1e-3,
              Cosmology(H0=_H0_EDS, Om_M=1.0), 0.02),
    2: Config(2, "lattice-32768-LCDM", 32768, 1, 0.05 / 32.0, _G_LCDM, 1000, 10, 1.37251071e-5,
              Cosmology(H0=70.0, Om_M=0.3, Om_L=0.7), 1.0 / 51.0,
              n_tracers=64, tracer_stride=512),
    3: Config(3, "plummer-131072-static", 131072, 2, 0.002, 1.0, 100, 10, 1e-3,
              None, 1.0, extra={"n_plummer": 91750, "b": 0.1}),
    4: Config(4, "clusters-2^20", 1 << 20, 3, 0.001, 1.0, 0, 0, 0.0, None, 1.0,
              oracle_targets=4096, extra={"n_clusters": 64, "sigma": 0.02}),
    5: Config(5, "clusters-2^22", 1 << 22, 4, 5e-4, 1.0, 0, 0, 0.0, None, 1.0,
              oracle_targets=4096, extra={"n_clusters": 256, "sigma": 0.02}),
}


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(seed))


def _uniform_cube(rng, n):
    return rng.random((n, 3))


def _lattice_jitter(rng, side, sigma_cells):
    g = (np.arange(side, dtype=np.float64) + 0.5) / side
    x, y, z = np.meshgrid(g, g, g, indexing="ij")
    p = np.stack([x.ravel(), y.ravel(), z.ravel()], axis=1)
    return p + rng.normal(0.0, sigma_cells / side, size=p.shape)


def _plummer_positions(rng, n, b, centre, r_max):
    """Plummer-profile radii r = b (u^{-2/3} - 1)^{-1/2}, isotropic directions,
    radii beyond r_max resampled."""
    r = np.empty(n)
    todo = np.arange(n)
    while todo.size:
        u = 1.0 - rng.random(todo.size)                 # (0, 1]
        rr = b / np.sqrt(np.maximum(u ** (-2.0 / 3.0) - 1.0, 1e-300))
        ok = rr <= r_max
        r[todo[ok]] = rr[ok]
        todo = todo[~ok]
    cos_t = 2.0 * rng.random(n) - 1.0
    phi = 2.0 * math.pi * rng.random(n)
    sin_t = np.sqrt(1.0 - cos_t * cos_t)
    d = np.stack([sin_t * np.cos(phi), sin_t * np.sin(phi), cos_t], axis=1)
    return centre + r[:, None] * d


def _clusters_plus_background(rng, n, n_clusters, sigma):
    n_cl = n // 2
    per = n_cl // n_clusters
    centres = rng.random((n_clusters, 3))
    cl = np.repeat(centres, per, axis=0) + rng.normal(0.0, sigma, size=(n_clusters * per, 3))
    bg = rng.random((n - n_clusters * per, 3))
    p = np.concatenate([cl, bg], axis=0)
    return p[rng.permutation(n)]


def _lognormal_masses(rng, n, sigma):
    m = np.exp(sigma * rng.standard_normal(n))
    return m / m.sum()


def make_config(index: int, n_override: int | None = None):
    """Return (cfg, pos_mass float32 [n,4], vel float32 [n,4]).

    `pos_mass[:, :3]` = comoving position, `pos_mass[:, 3]` = mass (layout D1,
    PAPER.md:123,135,142).  `vel[:, 3]` = 0.  `n_override` shrinks a config for
    quick tests while keeping its recipe (cluster/Plummer fractions scale).
    """
    cfg = CONFIGS[index]
    n = cfg.n if n_override is None else int(n_override)
    rng = _rng(cfg.seed)
    if index == 1:
        pos = _uniform_cube(rng, n)
        m = np.full(n, 1.0 / n)
    elif index == 2:
        side = round(n ** (1.0 / 3.0))
        if side ** 3 != n:
            raise ValueError("config 2 needs a cubic particle count")
        pos = _lattice_jitter(rng, side, 0.05)
        m = np.full(n, 1.0 / n)
    elif index == 3:
        n_pl = int(round(n * cfg.extra["n_plummer"] / cfg.n))
        pl = _plummer_positions(rng, n_pl, cfg.extra["b"], np.array([0.5, 0.5, 0.5]), 0.5)
        bg = _uniform_cube(rng, n - n_pl)
        pos = np.concatenate([pl, bg], axis=0)[rng.permutation(n)]
        m = np.full(n, 1.0 / n)
    elif index in (4, 5):
        ncl = cfg.extra["n_clusters"]
        if n_override is not None:
            ncl = max(1, min(ncl, n // 64))
        pos = _clusters_plus_background(rng, n, ncl, cfg.extra["sigma"])
        m = _lognormal_masses(rng, n, 0.5)
    else:
        raise KeyError(index)
    pos_mass = np.empty((n, 4), dtype=np.float32)
    pos_mass[:, :3] = pos.astype(np.float32)
    pos_mass[:, 3] = m.astype(np.float32)
    vel = np.zeros((n, 4), dtype=np.float32)
    if n_override is not None:
        cfg = Config(**{**cfg.__dict__, "n": n})
    return cfg, pos_mass, vel


def sample_targets(cfg: Config, n_targets: int | None = None) -> np.ndarray:
    """Seeded sample of target indices for the oracle check (configs 4, 5):
    the first `n_targets` entries of a permutation drawn with seed 1000+seed."""
    k = cfg.oracle_targets if n_targets is None else n_targets
    if k == 0 or k >= cfg.n:
        return np.arange(cfg.n, dtype=np.int64)
    return np.sort(_rng(1000 + cfg.seed).permutation(cfg.n)[:k]).astype(np.int64)


def tracer_indices(cfg: Config) -> np.ndarray:
    """Config 2: tracers are particles 512*t, t = 0..63 (G18)."""
    return (np.arange(cfg.n_tracers, dtype=np.int64) * cfg.tracer_stride).astype(np.int32)


def pack_pos_mass(pos: np.ndarray, m: np.ndarray) -> np.ndarray:
    """Assemble a float32 [n,4] body array from positions [n,3] and masses [n]."""
    out = np.empty((pos.shape[0], 4), dtype=np.float32)
    out[:, :3] = pos
    out[:, 3] = m
    return out
