"""Seeded synthetic inputs for the five BASELINE.json configs.

This module holds NO arithmetic of the method (no RHS, no stepper, no histogram): it only draws
masses, spin magnitudes and spin directions and packs them into the state layout
y = (omega, S1x,S1y,S1z, S2x,S2y,S2z, Lx,Ly,Lz).  It serves both the CUDA path and the oracle
(tests, bench.py), which is why it imports neither.

Recipe (paper: random initial spin orientations uniform on the sphere, L^ = (0,0,1), M = 1;
PAPER.md:68, 102-104): generator numpy Philox(seed); draws, each a length-N vector, in the fixed
order q, chi1, chi2, (z1, phi1), (z2, phi2); unit vectors from z = 2u-1, phi = 2 pi u' (exactly
uniform on the sphere; same distribution as the paper's Marsaglia sampler [21]);
m1 = 1/(1+q), m2 = q/(1+q); S_i = chi_i m_i^2 S^_i.
"""
from __future__ import annotations

from dataclasses import dataclass, replace

import numpy as np


@dataclass(frozen=True)
class Config:
    name: str
    n: int
    seed: int
    omega0: float
    omegaf: float
    q: tuple            # (lo, hi) for uniform q = m2/m1, or (q, q) fixed
    chi1: tuple         # (lo, hi) uniform, or fixed
    chi2: tuple
    s1_fixed_tilt_deg: float | None = None   # C4: S1 direction fixed, tilted from L^ in the x-z plane
    precision: str = "fp64"
    rtol: float = 1e-10
    atol: float = 1e-12
    bins: int = 50
    m1_fixed: float | None = None            # C4: m1 = 0.6, m2 = 0.4


CONFIGS = {
    # BASELINE.json configs[0..4]
    "C1": Config("C1", 1024, 0, 0.02, 0.05, (1.0, 1.0), (1.0, 1.0), (1.0, 1.0)),
    "C2": Config("C2", 1 << 20, 1, 0.005, 0.05, (1.0, 1.0), (1.0, 1.0), (1.0, 1.0)),
    "C3": Config("C3", 1 << 20, 2, 0.005, 0.05, (0.1, 1.0), (0.0, 1.0), (0.0, 1.0)),
    "C4": Config("C4", 1 << 22, 3, 0.01, 0.05, (0.4 / 0.6, 0.4 / 0.6), (0.9, 0.9), (1.0, 1.0),
                 s1_fixed_tilt_deg=60.0, m1_fixed=0.6),
    "C4f": Config("C4f", 1 << 22, 3, 0.01, 0.05, (0.4 / 0.6, 0.4 / 0.6), (0.9, 0.9), (1.0, 1.0),
                  s1_fixed_tilt_deg=60.0, m1_fixed=0.6, precision="fp32", rtol=1e-5, atol=1e-7),
    "C5": Config("C5", 1 << 18, 4, 0.001, 0.05, (0.25, 1.0), (0.0, 1.0), (0.0, 1.0)),
    # not a BASELINE.json config: C4 in mixed precision (float slopes, double state)
    "C4m": Config("C4m", 1 << 22, 3, 0.01, 0.05, (0.4 / 0.6, 0.4 / 0.6), (0.9, 0.9), (1.0, 1.0),
                  s1_fixed_tilt_deg=60.0, m1_fixed=0.6, precision="mixed", rtol=1e-7, atol=1e-9),
}


def with_size(cfg: Config, n: int) -> Config:
    """Same distribution and seed, first n systems (the draws are prefix-stable per column only
    for equal n, so a resized config is a different but identically distributed batch)."""
    return replace(cfg, n=int(n))


def _uniform(rng, lo_hi, n):
    lo, hi = lo_hi
    u = rng.random(n)          # always drawn, so the stream position does not depend on the config
    return lo + (hi - lo) * u if hi > lo else np.full(n, float(lo))


def _unit_vectors(rng, n):
    z = 2.0 * rng.random(n) - 1.0
    phi = 2.0 * np.pi * rng.random(n)
    r = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    return np.stack([r * np.cos(phi), r * np.sin(phi), z], axis=1)


def generate(cfg: Config):
    """Returns (init_states[n,10] float64, masses[n,2] float64)."""
    n = cfg.n
    rng = np.random.Generator(np.random.Philox(cfg.seed))
    q = _uniform(rng, cfg.q, n)
    chi1 = _uniform(rng, cfg.chi1, n)
    chi2 = _uniform(rng, cfg.chi2, n)
    s1hat = _unit_vectors(rng, n)
    s2hat = _unit_vectors(rng, n)
    if cfg.m1_fixed is not None:
        m1 = np.full(n, cfg.m1_fixed)
        m2 = 1.0 - m1
    else:
        m1 = 1.0 / (1.0 + q)
        m2 = q / (1.0 + q)
    if cfg.s1_fixed_tilt_deg is not None:
        th = np.deg2rad(cfg.s1_fixed_tilt_deg)
        s1hat = np.tile(np.array([np.sin(th), 0.0, np.cos(th)]), (n, 1))
    y0 = np.empty((n, 10))
    y0[:, 0] = cfg.omega0
    y0[:, 1:4] = (chi1 * m1 * m1)[:, None] * s1hat
    y0[:, 4:7] = (chi2 * m2 * m2)[:, None] * s2hat
    y0[:, 7:10] = np.array([0.0, 0.0, 1.0])
    masses = np.stack([m1, m2], axis=1)
    return np.ascontiguousarray(y0), np.ascontiguousarray(masses)


def philox_key(seed: int):
    """The Philox4x64 key numpy derives from an integer seed (SeedSequence): with it and counter 0 the raw
    stream of `np.random.Philox(seed)` is reproducible by any Philox4x64-10 implementation."""
    k = np.random.Philox(seed).state["state"]["key"]
    return int(k[0]), int(k[1])


def generator_spec(cfg: Config) -> dict:
    """The parameters of `generate(cfg)` in the form the on-device generator (pn_generate) and its oracle take."""
    return dict(key=philox_key(cfg.seed), omega0=cfg.omega0, q=cfg.q, chi1=cfg.chi1, chi2=cfg.chi2,
                m1_fixed=cfg.m1_fixed, s1_tilt_deg=cfg.s1_fixed_tilt_deg)


def sample_indices(n: int, k: int, seed: int = 12345) -> np.ndarray:
    """k distinct system indices of a batch of n (sorted), for sampled oracle comparisons."""
    rng = np.random.Generator(np.random.Philox(seed))
    k = min(k, n)
    return np.sort(rng.choice(n, size=k, replace=False))
