"""Seeded synthetic inputs for the open-boundary Poisson solve (numpy only).

This module is *data preparation*: it builds the charge-density meshes rho that
stand in for the OPAL cyclotron bunches of the paper's benchmark
(section 3.1.3 "similar problem setup as reported in [26, 27]";
mesh sizes PAPER.md:149-158, Table 1).  Those OPAL decks are not available, so
BASELINE.json's five configs are realised here as bunch-shaped particle clouds
deposited on the mesh with cloud-in-cell weights (recipe: SURVEY.md section 8(d),
restated in DESIGN.md "Input recipe").

It contains none of the method's arithmetic (no Green's function, no FFT, no
convolution) and is the only module shared by the CPU oracle's tests and the
CUDA path's tests/bench.  It imports neither of them.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Tuple

import numpy as np


@dataclass(frozen=True)
class Workload:
    """One BASELINE.json config: mesh n = (nx, ny, nz), spacing h = (hx, hy, hz) in metres."""

    name: str
    n: Tuple[int, int, int]          # (nx, ny, nz)  == paper's (Mx, My, Mz)
    h: Tuple[float, float, float]    # (hx, hy, hz)  [m]
    n_particles: int
    seed: int
    description: str


CONFIGS = (
    Workload("cfg1_16", (16, 16, 16), (1e-3, 1e-3, 1e-3), 10_000, 0,
             "16^3, 1e4 unit-charge particles, isotropic Gaussian sigma=3 cells"),
    Workload("cfg2_64", (64, 64, 64), (5e-4, 5e-4, 5e-4), 1_000_000, 1,
             "64^3, 1e6 particles, isotropic Gaussian sigma=8 cells, 1 nC"),
    Workload("cfg3_128", (128, 128, 128), (2e-4, 2e-4, 1e-4), 4_000_000, 2,
             "128^3, 4e6 particles, Gaussian sigma=(12,12,30) cells, 1 nC"),
    Workload("cfg4_256", (256, 256, 256), (1e-4, 1e-4, 1e-4), 16_000_000, 3,
             "256^3, 1.6e7 particles, uniform ellipsoid (80,80,110) + 5% halo sigma=20, 1 nC"),
    Workload("cfg5_64x64x512", (64, 64, 512), (3e-4, 3e-4, 5e-5), 8_000_000, 4,
             "64x64x512, 8e6 particles, transverse sigma=10, flat-top 400 with sigma=15 edges, 1 nC"),
)


def config(index_or_name) -> Workload:
    """Config by 1-based index (1..5, as BASELINE.json lists them) or by name."""
    if isinstance(index_or_name, int):
        return CONFIGS[index_or_name - 1]
    for w in CONFIGS:
        if w.name == index_or_name:
            return w
    raise KeyError(index_or_name)


def _positions_and_charge(w: Workload):
    """Particle positions in node-index units, shape (Np, 3) ordered (x, y, z), and charge per particle [C]."""
    rng = np.random.default_rng(w.seed)          # PCG64
    nx, ny, nz = w.n
    c = (np.array([nx, ny, nz], dtype=np.float64) - 1.0) / 2.0
    Np = w.n_particles
    if w.name == "cfg1_16":
        pos = c + 3.0 * rng.standard_normal((Np, 3))
        q = 1.0
    elif w.name == "cfg2_64":
        pos = c + 8.0 * rng.standard_normal((Np, 3))
        q = 1e-9 / Np
    elif w.name == "cfg3_128":
        pos = c + np.array([12.0, 12.0, 30.0]) * rng.standard_normal((Np, 3))
        q = 1e-9 / Np
    elif w.name == "cfg4_256":
        n_core = (Np * 95) // 100
        n_halo = Np - n_core
        d = rng.standard_normal((n_core, 3))
        d /= np.sqrt((d * d).sum(axis=1, keepdims=True))
        r = rng.random(n_core) ** (1.0 / 3.0)
        core = c + (d * r[:, None]) * np.array([80.0, 80.0, 110.0])
        halo = c + 20.0 * rng.standard_normal((n_halo, 3))
        pos = np.concatenate([core, halo], axis=0)
        q = 1e-9 / Np
    elif w.name == "cfg5_64x64x512":
        xy = c[:2] + 10.0 * rng.standard_normal((Np, 2))
        u = rng.random(Np)
        z = c[2] + (400.0 * u - 200.0) + 15.0 * rng.standard_normal(Np)
        pos = np.concatenate([xy, z[:, None]], axis=1)
        q = 1e-9 / Np
    else:
        raise KeyError(w.name)
    return pos, q


def cic_deposit(pos: np.ndarray, q: float, n, h) -> np.ndarray:
    """Cloud-in-cell deposit onto rho[nz][ny][nx] (x fastest), in C/m^3.

    A particle is dropped unless 0 <= pos < n-1 on every axis; q is fixed before dropping.
    """
    nx, ny, nz = n
    hx, hy, hz = h
    lim = np.array([nx - 1, ny - 1, nz - 1], dtype=np.float64)
    keep = np.all((pos >= 0.0) & (pos < lim), axis=1)
    p = pos[keep]
    i0 = np.floor(p).astype(np.int64)
    f = p - i0
    rho = np.zeros(nx * ny * nz, dtype=np.float64)
    for dz in (0, 1):
        wz = f[:, 2] if dz else 1.0 - f[:, 2]
        for dy in (0, 1):
            wy = f[:, 1] if dy else 1.0 - f[:, 1]
            for dx in (0, 1):
                wx = f[:, 0] if dx else 1.0 - f[:, 0]
                lin = ((i0[:, 2] + dz) * ny + (i0[:, 1] + dy)) * nx + (i0[:, 0] + dx)
                rho += np.bincount(lin, weights=wx * wy * wz, minlength=rho.size)
    rho *= q / (hx * hy * hz)
    return rho.reshape(nz, ny, nx)


def particles(w: Workload, origin=None, count=None):
    """The config's particles as physical coordinates x, y, z [m] (node (i, j, k) sits at origin + (i hx, j hy, k hz);
    default origin: the mesh centred on 0) and charges q [C]: four float64 arrays.  `count` keeps the first particles only."""
    pos, q = _positions_and_charge(w)
    if count is not None:
        pos = pos[:count]
    h = np.array(w.h, dtype=np.float64)
    if origin is None:
        origin = -0.5 * (np.array(w.n, dtype=np.float64) - 1.0) * h
    origin = np.asarray(origin, dtype=np.float64)
    xyz = origin + pos * h
    return (np.ascontiguousarray(xyz[:, 0]), np.ascontiguousarray(xyz[:, 1]), np.ascontiguousarray(xyz[:, 2]),
            np.full(len(pos), q, dtype=np.float64), tuple(float(v) for v in origin))


def make_rho(w: Workload) -> np.ndarray:
    """The config's charge density, contiguous float64 [nz][ny][nx]."""
    pos, q = _positions_and_charge(w)
    return np.ascontiguousarray(cic_deposit(pos, q, w.n, w.h))


def random_rho(n, seed: int, signed: bool = True) -> np.ndarray:
    """Small generic test field: iid values on [nz][ny][nx] (for edge-case and invariant tests)."""
    nx, ny, nz = n
    rng = np.random.default_rng(seed)
    a = rng.standard_normal((nz, ny, nx)) if signed else rng.random((nz, ny, nx))
    return np.ascontiguousarray(a)


def sample_nodes(n, seed: int, count: int = 64) -> np.ndarray:
    """Output nodes for sampled checks: `count` seeded random nodes + 8 corners + centre; rows are (i, j, k) = (x, y, z)."""
    nx, ny, nz = n
    rng = np.random.default_rng(1000 + seed)
    r = np.stack([rng.integers(0, nx, count), rng.integers(0, ny, count), rng.integers(0, nz, count)], axis=1)
    corners = np.array([[i, j, k] for k in (0, nz - 1) for j in (0, ny - 1) for i in (0, nx - 1)])
    centre = np.array([[nx // 2, ny // 2, nz // 2]])
    return np.concatenate([r, corners, centre], axis=0).astype(np.int64)
