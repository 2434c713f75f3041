"""Seeded synthetic inputs shared by the tests, the oracle harness and bench.py.

This module holds NONE of the method's arithmetic (no basis functions, no quadrature,
no operator): only the counter-based uniform generator of SURVEY.md §8(d), the five
workload configurations of BASELINE.json, and the perturbed-vertex recipe of config 3
(SURVEY.md §8(c) reading 5).  Both the CPU oracle's callers and the CUDA path's callers
take their X / vertices from here, so the two sides see bit-identical inputs.

Generator:
    u(seed, k) = 2 * ((splitmix64(seed + k*0x9E3779B97F4A7C15) >> 11) * 2^-53) - 1
with k the linear element index.  The library's device-side `fe_fill_uniform` implements
the same function (it is an input generator, not part of the operator) and is tested
bit-exact against `uniform_pm1` below.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional, Tuple

import numpy as np

GOLDEN = np.uint64(0x9E3779B97F4A7C15)
SEED_BASE = 220807129 * 10  # X of config c -> SEED_BASE + c

BC_PERIODIC = 0
BC_DIRICHLET = 1
GEOM_AFFINE = 0
GEOM_QPOINT = 1


def splitmix64(z: np.ndarray) -> np.ndarray:
    """Finaliser of SplitMix64 on a uint64 array (wrap-around arithmetic)."""
    z = z.astype(np.uint64, copy=True)
    with np.errstate(over="ignore"):
        z ^= z >> np.uint64(30)
        z *= np.uint64(0xBF58476D1CE4E5B9)
        z ^= z >> np.uint64(27)
        z *= np.uint64(0x94D049BB133111EB)
        z ^= z >> np.uint64(31)
    return z


def uniform_pm1(seed: int, start: int, count: int) -> np.ndarray:
    """u(seed, k) for k = start .. start+count-1, float64 in [-1, 1)."""
    k = np.arange(start, start + count, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = np.uint64(seed) + k * GOLDEN
    h = splitmix64(z) >> np.uint64(11)
    return 2.0 * (h.astype(np.float64) * 2.0 ** -53) - 1.0


def multivector(seed: int, ndof: int, nvec: int, rows: Optional[np.ndarray] = None) -> np.ndarray:
    """X[J, beta] = u(seed, J*nvec + beta), shape (ndof, nvec); `rows` selects a subset of J."""
    if rows is None:
        return uniform_pm1(seed, 0, ndof * nvec).reshape(ndof, nvec)
    rows = np.asarray(rows, dtype=np.uint64)
    k = (rows[:, None] * np.uint64(nvec) + np.arange(nvec, dtype=np.uint64)[None, :]).ravel()
    with np.errstate(over="ignore"):
        z = np.uint64(seed) + k * GOLDEN
    h = splitmix64(z) >> np.uint64(11)
    return (2.0 * (h.astype(np.float64) * 2.0 ** -53) - 1.0).reshape(len(rows), nvec)


@dataclass(frozen=True)
class Workload:
    """One BASELINE.json configuration (mesh + operator + multivector shape)."""
    name: str
    p: int
    ncells: Tuple[int, int, int]
    bc: int
    geom: int
    sigma: float
    box_lo: Tuple[float, float, float]
    box_hi: Tuple[float, float, float]
    nvec: int
    seed: int
    perturb: float = 0.0          # fraction of h by which interior vertices move (config 3)
    cheb_m: int = 0               # Chebyshev degree (config 5)
    cheb_a: float = 0.0
    cheb_a0: float = 0.0
    nvec_sweep: Tuple[int, ...] = field(default_factory=tuple)

    @property
    def nd(self) -> Tuple[int, int, int]:
        add = 1 if self.bc == BC_DIRICHLET else 0
        return tuple(n * self.p + add for n in self.ncells)

    @property
    def ndof(self) -> int:
        nd = self.nd
        return nd[0] * nd[1] * nd[2]

    def scaled(self, ncells: int, nvec: Optional[int] = None) -> "Workload":
        """Same recipe on a smaller mesh (parity-test sizes); the box keeps h fixed."""
        h = [(hi - lo) / n for lo, hi, n in zip(self.box_lo, self.box_hi, self.ncells)]
        hi = tuple(lo + hh * ncells for lo, hh in zip(self.box_lo, h))
        return Workload(self.name + f"@{ncells}", self.p, (ncells,) * 3, self.bc, self.geom, self.sigma,
                        self.box_lo, hi, self.nvec if nvec is None else nvec, self.seed,
                        self.perturb, self.cheb_m, self.cheb_a, self.cheb_a0, self.nvec_sweep)


def configs() -> dict:
    """The five BASELINE.json configurations (SURVEY.md §8 'Sizes at BASELINE.json's configs')."""
    z3, o3, t3 = (0.0, 0.0, 0.0), (1.0, 1.0, 1.0), (10.0, 10.0, 10.0)
    return {
        1: Workload("cfg1_p4_periodic_8c", 4, (8, 8, 8), BC_PERIODIC, GEOM_AFFINE, 1.0, z3, o3, 8, SEED_BASE + 1),
        2: Workload("cfg2_p6_dirichlet_24c", 6, (24, 24, 24), BC_DIRICHLET, GEOM_AFFINE, 0.5, z3, t3, 32, SEED_BASE + 2),
        3: Workload("cfg3_p8_periodic_16c_perturbed", 8, (16, 16, 16), BC_PERIODIC, GEOM_QPOINT, 1.0, z3, o3, 16,
                    SEED_BASE + 3, perturb=0.15),
        4: Workload("cfg4_p7_periodic_32c", 7, (32, 32, 32), BC_PERIODIC, GEOM_AFFINE, 1.0, z3, o3, 64, SEED_BASE + 4,
                    nvec_sweep=(1, 8, 16, 32, 64)),
        # SURVEY.md §8(c) reading 12: config 5 lives on [0,10]^3 so that [2.0, b] is a valid interval.
        5: Workload("cfg5_p6_periodic_16c_cheb20", 6, (16, 16, 16), BC_PERIODIC, GEOM_AFFINE, 1.0, z3, t3, 1024,
                    SEED_BASE + 5, cheb_m=20, cheb_a=2.0, cheb_a0=0.0),
    }


def uniform_vertices(ncells, box_lo, box_hi) -> np.ndarray:
    """Vertex array [(ncz+1)][(ncy+1)][(ncx+1)][3] of the uniform Cartesian mesh."""
    ncx, ncy, ncz = ncells
    xs = [np.linspace(box_lo[d], box_hi[d], n + 1) for d, n in enumerate((ncx, ncy, ncz))]
    v = np.empty((ncz + 1, ncy + 1, ncx + 1, 3), dtype=np.float64)
    v[..., 0] = xs[0][None, None, :]
    v[..., 1] = xs[1][None, :, None]
    v[..., 2] = xs[2][:, None, None]
    return v


def perturbed_vertices(ncells, box_lo, box_hi, frac: float, seed: int) -> np.ndarray:
    """Config-3 mesh (SURVEY.md §8(c) reading 5): vertex (i,j,k) moves iff it is strictly inside the
    box in every direction; each coordinate gets an independent draw in [-frac*h, frac*h] with
    k = ((kz*(ncy+1)+ky)*(ncx+1)+kx)*3 + comp of the counter generator."""
    ncx, ncy, ncz = ncells
    v = uniform_vertices(ncells, box_lo, box_hi)
    u = uniform_pm1(seed, 0, v.size).reshape(v.shape)
    h = np.array([(box_hi[d] - box_lo[d]) / n for d, n in enumerate((ncx, ncy, ncz))])
    interior = np.zeros(v.shape[:3], dtype=bool)
    interior[1:ncz, 1:ncy, 1:ncx] = True
    v += np.where(interior[..., None], u * (frac * h)[None, None, None, :], 0.0)
    return v


def workload_vertices(w: Workload) -> Optional[np.ndarray]:
    """Explicit vertex array for per-q-point geometry workloads, None for uniform Cartesian."""
    if w.geom == GEOM_QPOINT:
        return perturbed_vertices(w.ncells, w.box_lo, w.box_hi, w.perturb, w.seed + 100)
    return None


def kappa_points(seed: int, ncells: int, n3: int, lo: float = -1.0, hi: float = 3.0) -> np.ndarray:
    """Synthetic stand-in for the 'precomputed potential' kappa of PAPER.md:796: one value per quadrature point,
    [ncells][n3], independent draws in [lo, hi] from the counter generator (the kernels' cost does not depend on the
    values; smooth potentials are built in the tests from the oracle's quadrature-point coordinates)."""
    u = uniform_pm1(seed, 0, ncells * n3).reshape(ncells, n3)
    return lo + (hi - lo) * 0.5 * (u + 1.0)
