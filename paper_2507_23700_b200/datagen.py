"""Seeded synthetic input generators (BASELINE.json configs C1..C5 and small test shapes).

This module holds NONE of the method's arithmetic: it only draws seeded random fp32
arrays (numpy PCG64; sample in fp64, round once to fp32 -- SURVEY.md §8(d), reading A22).
It serves both the oracle-side tests and the CUDA-side tests/bench, and imports neither.

Layouts (row-major fp32), matching include/arbx.h:
  POINT  : (n, D)            coordinates
  BOX    : (n, 2D)           lo[D] then hi[D]
  SPHERE : (n, D+1)          centre[D] then radius
"""
from __future__ import annotations

import math
import numpy as np

POINT, BOX, SPHERE = 0, 1, 2

__all__ = [
    "POINT", "BOX", "SPHERE", "rng", "uniform_points", "uniform_boxes", "uniform_spheres",
    "sphere_queries", "config", "CONFIG_NAMES", "radius_for_expected", "lattice_points",
    "lattice_cells", "gaussian_mixture",
]


def rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(seed))


def uniform_points(n: int, dim: int, seed: int, scale: float = 1.0) -> np.ndarray:
    g = rng(seed)
    return (scale * g.random((n, dim))).astype(np.float32)


def uniform_boxes(n: int, dim: int, seed: int, h: float) -> np.ndarray:
    """Centres U[0,1)^D, per-axis half-widths U[0.5h,1.5h) (BASELINE.json configs[3])."""
    g = rng(seed)
    c = g.random((n, dim))
    w = h * (0.5 + g.random((n, dim)))
    lo = (c - w).astype(np.float32)
    hi = (c + w).astype(np.float32)
    return np.concatenate([lo, np.maximum(lo, hi)], axis=1)


def uniform_spheres(n: int, dim: int, seed: int, rmax: float) -> np.ndarray:
    g = rng(seed)
    c = g.random((n, dim))
    r = rmax * (0.25 + 0.75 * g.random((n, 1)))
    return np.concatenate([c, r], axis=1).astype(np.float32)


def sphere_queries(points: np.ndarray, r: float) -> np.ndarray:
    """Attach one radius to every query point -> SPHERE layout (centre, r)."""
    q = np.empty((points.shape[0], points.shape[1] + 1), dtype=np.float32)
    q[:, :-1] = points
    q[:, -1] = np.float32(r)
    return q


def radius_for_expected(m: float, density: float, dim: int = 3) -> float:
    """Radius of the D-ball holding m points at the given density (r = (m/(rho V_D))^(1/D))."""
    vd = math.pi ** (dim / 2) / math.gamma(dim / 2 + 1)
    return (m / (density * vd)) ** (1.0 / dim)


def lattice_points(g: int, dim: int) -> np.ndarray:
    """Integer lattice {0..g-1}^D as fp32 points (closed-form pins P2/P2')."""
    axes = [np.arange(g, dtype=np.float32)] * dim
    return np.stack(np.meshgrid(*axes, indexing="ij"), axis=-1).reshape(-1, dim).copy()


def lattice_cells(g: int, dim: int) -> np.ndarray:
    """Unit cells [z,z+1]^D as BOX primitives (pin P3)."""
    lo = lattice_points(g, dim)
    return np.concatenate([lo, lo + 1.0], axis=1).astype(np.float32)


def gaussian_mixture(n: int, dim: int, seed: int, centre_seed: int = 2, ncomp: int = 64,
                     sigma: float = 0.02) -> np.ndarray:
    """Equal-weight isotropic Gaussian mixture clipped to [0,1] (BASELINE.json configs[4])."""
    centres = rng(centre_seed).random((ncomp, dim))
    g = rng(seed)
    comp = g.integers(0, ncomp, size=n)
    x = centres[comp] + sigma * g.standard_normal((n, dim))
    return np.clip(x, 0.0, 1.0).astype(np.float32)


CONFIG_NAMES = ("C1", "C2", "C3", "C4", "C5")


def config(name: str, scale: float = 1.0, seed_offset: int = 0) -> dict:
    """The five BASELINE.json workloads. `scale` < 1 shrinks N and Q (same law, same density
    relations) for quick parity cases; scale == 1 is the size BASELINE.json states.
    `seed_offset` shifts the data/query seeds (0, 1) so that bench.py replicas draw distinct
    inputs of the same law; the parity tests always use offset 0.

    Returns dict(prims, pkind, dim, queries (spatial layout), qkind, qpoints (kNN) or None,
                 k or None, r or None, name, n, nq).
    """
    s0, s1 = seed_offset, seed_offset + 1
    if name == "C1":
        n = nq = max(1, int(10_000 * scale))
        p = uniform_points(n, 3, s0)
        qp = uniform_points(nq, 3, s1)
        r = 0.0620
        return dict(name=name, prims=p, pkind=POINT, dim=3, queries=sphere_queries(qp, r),
                    qkind=SPHERE, qpoints=qp, k=10, r=r, n=n, nq=nq)
    if name == "C2":
        n = nq = max(1, int(1_000_000 * scale))
        p = uniform_points(n, 3, s0)
        qp = uniform_points(nq, 3, s1)
        r = radius_for_expected(16.0, float(n), 3)
        return dict(name=name, prims=p, pkind=POINT, dim=3, queries=sphere_queries(qp, r),
                    qkind=SPHERE, qpoints=qp, k=None, r=r, n=n, nq=nq)
    if name == "C3":
        n = nq = max(1, int(10_000_000 * scale))
        a = float(n) ** (1.0 / 3.0)
        p = uniform_points(n, 3, s0, scale=a)
        g = rng(s1)
        v = g.standard_normal((nq, 3))
        v /= np.linalg.norm(v, axis=1, keepdims=True)
        qp = (0.5 * a + 0.5 * a * v).astype(np.float32)
        r = radius_for_expected(16.0, 1.0, 3)
        return dict(name=name, prims=p, pkind=POINT, dim=3, queries=sphere_queries(qp, r),
                    qkind=SPHERE, qpoints=qp, k=16, r=r, n=n, nq=nq)
    if name == "C4":
        n = max(1, int(10_000_000 * scale))
        nq = max(1, int(5_000_000 * scale))
        h = 0.5 * float(n) ** (-1.0 / 3.0)
        p = uniform_boxes(n, 3, s0, h)
        q = uniform_boxes(nq, 3, s1, 2.0 * h)
        return dict(name=name, prims=p, pkind=BOX, dim=3, queries=q, qkind=BOX,
                    qpoints=None, k=None, r=None, n=n, nq=nq)
    if name == "C5":
        n = max(1, int(4_000_000 * scale))
        nq = max(1, int(1_000_000 * scale))
        p = gaussian_mixture(n, 5, s0)
        qp = gaussian_mixture(nq, 5, s1)
        r = 0.01
        return dict(name=name, prims=p, pkind=POINT, dim=5, queries=sphere_queries(qp, r),
                    qkind=SPHERE, qpoints=qp, k=8, r=r, n=n, nq=nq)
    raise ValueError(f"unknown config {name!r}")
