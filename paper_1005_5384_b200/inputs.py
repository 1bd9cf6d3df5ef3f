"""Seeded synthetic workloads (BASELINE.json `configs`).

This module is the ONLY code shared by the oracle (`oracle/`) and the CUDA path
(`paper_1005_5384_b200/csrc/`).  It holds none of the method's arithmetic: it
only draws particle positions / masses / velocities.  It depends on numpy alone
and never imports the CUDA binding or the oracle.

The paper's own workload is a Milky-Way bulge/disk/halo model (PAPER.md:145,
ref [21]); that generator is not available, so Plummer spheres (centrally
concentrated) and a uniform cube (low contrast) stand in for it, as
BASELINE.json prescribes.

All recipes use ``numpy.random.Generator(numpy.random.PCG64(seed))`` and draw in
a fixed order, so a (name, n, seed) triple always yields bit-identical fp32
arrays.
"""
from __future__ import annotations

import numpy as np

#: mass fraction of a Plummer sphere inside r = 10 a:  10^3 / 101^(3/2)
PLUMMER_X_MAX = 1000.0 / 101.0 ** 1.5


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(seed))


def plummer_positions64(n: int, seed: int, a: float = 1.0) -> np.ndarray:
    """fp64 positions of a Plummer sphere of scale radius ``a`` truncated at 10 a.

    Recipe: U1, U2, U3 = rng.random(n) three times in that
    order; enclosed-mass fraction X = U1 * X_max (CDF truncation, no
    rejection), clamped to >= 1e-12; r = a (X^(-2/3) - 1)^(-1/2);
    cos(theta) = 2 U2 - 1; phi = 2 pi U3.
    """
    rng = _rng(seed)
    u1 = rng.random(n)
    u2 = rng.random(n)
    u3 = rng.random(n)
    x = np.maximum(u1 * PLUMMER_X_MAX, 1e-12)
    r = a / np.sqrt(x ** (-2.0 / 3.0) - 1.0)
    ct = 2.0 * u2 - 1.0
    st = np.sqrt(np.maximum(0.0, 1.0 - ct * ct))
    ph = 2.0 * np.pi * u3
    return np.stack([r * st * np.cos(ph), r * st * np.sin(ph), r * ct], axis=1)


def plummer(n: int, seed: int, a: float = 1.0):
    """(pos fp32 [n,3], mass fp32 [n]) — equal masses 1/n, G = 1."""
    pos = plummer_positions64(n, seed, a).astype(np.float32)
    mass = np.full(n, 1.0 / n, dtype=np.float32)
    return np.ascontiguousarray(pos), mass


def uniform_cube(n: int, seed: int):
    """Uniform random cube [-1,1]^3, equal masses 1/n (config 2, low contrast)."""
    rng = _rng(seed)
    pos = rng.uniform(-1.0, 1.0, (n, 3)).astype(np.float32)
    mass = np.full(n, 1.0 / n, dtype=np.float32)
    return np.ascontiguousarray(pos), mass


def plummer_velocities64(pos64_rel: np.ndarray, seed: int, mtot: float, a: float) -> np.ndarray:
    """Isotropic Plummer velocities (Aarseth-Henon-Wielen rejection), G = 1.

    q drawn with density q^2 (1-q^2)^(7/2) by rejection against 0.1;
    v = q * sqrt(2 M / a) * (1 + (r/a)^2)^(-1/4).  Harness-only (config 5);
    the force path never sees velocities.
    """
    rng = _rng(seed)
    n = pos64_rel.shape[0]
    q = np.empty(n)
    todo = np.arange(n)
    while todo.size:
        x = rng.random(todo.size)
        y = rng.random(todo.size) * 0.1
        ok = y < x * x * (1.0 - x * x) ** 3.5
        q[todo[ok]] = x[ok]
        todo = todo[~ok]
    r2 = (pos64_rel ** 2).sum(1) / (a * a)
    v = q * np.sqrt(2.0 * mtot / a) * (1.0 + r2) ** -0.25
    ct = 2.0 * rng.random(n) - 1.0
    st = np.sqrt(np.maximum(0.0, 1.0 - ct * ct))
    ph = 2.0 * np.pi * rng.random(n)
    return np.stack([v * st * np.cos(ph), v * st * np.sin(ph), v * ct], axis=1)


def two_plummer(n_total: int, seed1: int = 5, seed2: int = 6, with_velocities: bool = False):
    """Config 5: two offset Plummer spheres, mass ratio 3:1, equal particle masses.

    N1 = 3N/4 (M1 = 0.75, a = 1) centred at x = -1.5 moving at +0.125;
    N2 = N/4  (M2 = 0.25, a = 0.5) centred at x = +4.5 moving at -0.375
    (centres 6 apart, COM at origin, closing speed 0.5, zero net momentum).
    Returns (pos fp32, mass fp32) or (pos, mass, vel fp32).
    """
    n1 = (3 * n_total) // 4
    n2 = n_total - n1
    p1 = plummer_positions64(n1, seed1, 1.0)
    p2 = plummer_positions64(n2, seed2, 0.5)
    pos = np.concatenate([p1 + np.array([-1.5, 0.0, 0.0]), p2 + np.array([4.5, 0.0, 0.0])])
    mass = np.full(n_total, 1.0 / n_total, dtype=np.float32)
    pos32 = np.ascontiguousarray(pos.astype(np.float32))
    if not with_velocities:
        return pos32, mass
    v1 = plummer_velocities64(p1, seed1 + 100, 0.75, 1.0) + np.array([0.125, 0.0, 0.0])
    v2 = plummer_velocities64(p2, seed2 + 100, 0.25, 0.5) + np.array([-0.375, 0.0, 0.0])
    vel = np.concatenate([v1, v2]).astype(np.float32)
    return pos32, mass, np.ascontiguousarray(vel)


def sample_targets(n: int, k: int, seed: int = 4) -> np.ndarray:
    """Config 4: k particle indices without replacement (sorted), rng(seed).choice."""
    idx = _rng(seed).choice(n, size=min(k, n), replace=False)
    return np.sort(idx).astype(np.int64)


WORKLOADS = {
    # name: (callable, kwargs, theta, eps, n_leaf)  -- BASELINE.json configs[0..4]
    "plummer_1k": (plummer, dict(n=1024, seed=1), 0.5, 0.01, 16),
    "plummer_64k": (plummer, dict(n=65536, seed=2), 0.5, 0.01, 16),
    "cube_64k": (uniform_cube, dict(n=65536, seed=2), 0.5, 0.01, 16),
    "plummer_1m": (plummer, dict(n=1 << 20, seed=3), 0.5, 0.01, 16),
    "two_plummer_16m": (two_plummer, dict(n_total=1 << 24), 0.5, 0.005, 16),
}


def make(name: str):
    """Return (pos, mass, theta, eps, n_leaf) for a named BASELINE.json workload."""
    fn, kw, theta, eps, n_leaf = WORKLOADS[name]
    pos, mass = fn(**kw)[:2]
    return pos, mass, theta, eps, n_leaf
