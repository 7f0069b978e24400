"""Analytic magnetic fields sampled on rectilinear grids (data only).

Array layout everywhere: C-contiguous numpy arrays of shape (nz, ny, nx), i.e.
flat index (k*ny + j)*nx + i with x fastest.  Grids are node-sampled: node i
of axis d sits at lo_d + i*(hi_d - lo_d)/(n_d - 1) (uniform) or at the given
coordinate array (stretched).  Fields are evaluated in fp64; rounding to the
storage type is done by whoever packs the field (oracle O0 / qsl_field_create).
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

from .rng import SplitMix64


@dataclasses.dataclass
class Grid:
    """Rectilinear node grid.  `xs, ys, zs` are always filled (fp64 node coordinates)."""
    nx: int
    ny: int
    nz: int
    lo: tuple
    hi: tuple
    stretched: bool
    xs: np.ndarray
    ys: np.ndarray
    zs: np.ndarray

    @staticmethod
    def uniform(n, lo, hi) -> "Grid":
        nx, ny, nz = n
        ax = []
        for d, nd in enumerate((nx, ny, nz)):
            h = (hi[d] - lo[d]) / (nd - 1)
            ax.append(lo[d] + np.arange(nd, dtype=np.float64) * h)
        return Grid(nx, ny, nz, tuple(map(float, lo)), tuple(map(float, hi)), False, *ax)

    @staticmethod
    def from_axes(xs, ys, zs) -> "Grid":
        xs, ys, zs = (np.ascontiguousarray(a, dtype=np.float64) for a in (xs, ys, zs))
        return Grid(len(xs), len(ys), len(zs), (xs[0], ys[0], zs[0]), (xs[-1], ys[-1], zs[-1]), True, xs, ys, zs)

    @property
    def shape(self):
        return (self.nz, self.ny, self.nx)

    @property
    def n_nodes(self):
        return self.nx * self.ny * self.nz


def stretched_axis(n: int, lo: float, hi: float, ratio: float) -> np.ndarray:
    """Geometrically stretched node coordinates: cell widths grow by `ratio` from first to last cell."""
    if n < 2:
        raise ValueError("need >= 2 nodes")
    w = ratio ** (np.arange(n - 1, dtype=np.float64) / max(n - 2, 1))
    x = np.concatenate([[0.0], np.cumsum(w)])
    x = lo + (hi - lo) * x / x[-1]
    x[0], x[-1] = lo, hi
    return x


def _mesh(grid: Grid):
    Z, Y, X = np.meshgrid(grid.zs, grid.ys, grid.xs, indexing="ij")
    return X, Y, Z


def uniform_field(grid: Grid, direction):
    """B = const vector `direction` (pin P1: Q = 2)."""
    d = np.asarray(direction, dtype=np.float64)
    return tuple(np.full(grid.shape, d[c], dtype=np.float64) for c in range(3))


def hyperbolic_B(points: np.ndarray, k: float) -> np.ndarray:
    """B = (k x, -k y, 1) at arbitrary points (n,3)."""
    p = np.asarray(points, dtype=np.float64)
    return np.stack([k * p[:, 0], -k * p[:, 1], np.ones(len(p))], axis=1)


def hyperbolic_field(grid: Grid, k: float):
    """B = (k x, -k y, 1) on the grid (config 1; BASELINE.json configs[0])."""
    X, Y, _ = _mesh(grid)
    return (np.ascontiguousarray(k * X), np.ascontiguousarray(-k * Y), np.ones(grid.shape, dtype=np.float64))


def quadrupole_charges(seed: int = 160900724, shift=(0.0, 0.0), depth: float = 0.1):
    """Four sub-photospheric charges q=(+1,-1,+1,-1) at x=(-0.3,-0.1,0.1,0.3), y_i ~ U(-0.05,0.05), z=-depth.

    BASELINE.json configs[1]; reading A13 (y-offsets uniform in +-0.05 from the D0 RNG).
    Returns (q[4], r[4,3]).
    """
    rng = SplitMix64(seed)
    q = np.array([1.0, -1.0, 1.0, -1.0])
    xs = np.array([-0.3, -0.1, 0.1, 0.3])
    ys = np.array([rng.uniform(-0.05, 0.05) for _ in range(4)])
    r = np.stack([xs + shift[0], ys + shift[1], np.full(4, -depth)], axis=1)
    return q, r


def quadrupole_B(points: np.ndarray, q: np.ndarray, r: np.ndarray) -> np.ndarray:
    """B = sum_i q_i (x - r_i)/|x - r_i|^3 at arbitrary points (n,3)."""
    p = np.asarray(points, dtype=np.float64)
    out = np.zeros_like(p)
    for qi, ri in zip(q, r):
        d = p - ri[None, :]
        out += qi * d / (np.sum(d * d, axis=1) ** 1.5)[:, None]
    return out


def quadrupole_field(grid: Grid, q: np.ndarray, r: np.ndarray):
    """Potential field of point charges on the grid, evaluated plane by plane to bound memory."""
    bx = np.zeros(grid.shape); by = np.zeros(grid.shape); bz = np.zeros(grid.shape)
    Y, X = np.meshgrid(grid.ys, grid.xs, indexing="ij")
    for k, z in enumerate(grid.zs):
        for qi, ri in zip(q, r):
            dx = X - ri[0]; dy = Y - ri[1]; dz = z - ri[2]
            inv = qi / (dx * dx + dy * dy + dz * dz) ** 1.5
            bx[k] += dx * inv; by[k] += dy * inv; bz[k] += dz * inv
    return bx, by, bz


def lfff_modes(seed: int = 160900725, n_modes: int = 32, alpha: float = 1.5):
    """Mode table of the linear force-free field (BASELINE.json configs[3]).

    Per mode, in this draw order: |k| = 2pi + 6pi*u01, psi = 2pi*u01, phi = 2pi*u01;
    kx = |k| cos psi, ky = |k| sin psi, l = sqrt(k^2 - alpha^2), A = |k|^-1.5.
    """
    rng = SplitMix64(seed)
    km = np.empty(n_modes); psi = np.empty(n_modes); phi = np.empty(n_modes)
    for m in range(n_modes):
        km[m] = 2 * math.pi + 6 * math.pi * rng.u01()
        psi[m] = 2 * math.pi * rng.u01()
        phi[m] = 2 * math.pi * rng.u01()
    kx = km * np.cos(psi); ky = km * np.sin(psi)
    l = np.sqrt(km * km - alpha * alpha)
    A = km ** -1.5
    return dict(alpha=alpha, kmag=km, kx=kx, ky=ky, l=l, A=A, phi=phi)


def lfff_B(points: np.ndarray, modes: dict) -> np.ndarray:
    """LFFF at arbitrary points: Bz = A cos(th) e^{-lz}, Bx = A (l kx - a ky)/k^2 sin(th) e^{-lz}, By likewise."""
    p = np.asarray(points, dtype=np.float64)
    kx, ky, l, A, phi, km, a = (modes[n] for n in ("kx", "ky", "l", "A", "phi", "kmag", "alpha"))
    th = np.outer(p[:, 0], kx) + np.outer(p[:, 1], ky) + phi[None, :]
    e = np.exp(-np.outer(p[:, 2], l))
    cx = A * (l * kx - a * ky) / km ** 2
    cy = A * (l * ky + a * kx) / km ** 2
    s = np.sin(th) * e
    return np.stack([(cx * s).sum(1), (cy * s).sum(1), (A * np.cos(th) * e).sum(1)], axis=1)


def lfff_field(grid: Grid, modes: dict):
    """LFFF on the grid; separable in (x,y) and z, so cost is modes * (nx*ny + nz) transcendental calls."""
    kx, ky, l, A, phi, km, a = (modes[n] for n in ("kx", "ky", "l", "A", "phi", "kmag", "alpha"))
    Y, X = np.meshgrid(grid.ys, grid.xs, indexing="ij")
    bx = np.zeros(grid.shape); by = np.zeros(grid.shape); bz = np.zeros(grid.shape)
    for m in range(len(kx)):
        th = kx[m] * X + ky[m] * Y + phi[m]
        s = np.sin(th); c = np.cos(th)
        ez = np.exp(-l[m] * grid.zs)[:, None, None]
        cxm = A[m] * (l[m] * kx[m] - a * ky[m]) / km[m] ** 2
        cym = A[m] * (l[m] * ky[m] + a * kx[m]) / km[m] ** 2
        bx += cxm * s[None] * ez
        by += cym * s[None] * ez
        bz += A[m] * c[None] * ez
    return bx, by, bz


def superposition_field(grid: Grid, q, r, modes, rel_amp: float = 0.1):
    """B = B_quad + w * B_lfff with w such that rms|B_lfff| = rel_amp * rms|B_quad| over the z = zs[0] node plane.

    Reading A12 (BASELINE.json configs[4] gives no relative weight).  Returns (bx, by, bz, w).
    """
    qx, qy, qz = quadrupole_field(grid, q, r)
    lx, ly, lz = lfff_field(grid, modes)
    rq = math.sqrt(float(np.mean(qx[0] ** 2 + qy[0] ** 2 + qz[0] ** 2)))
    rl = math.sqrt(float(np.mean(lx[0] ** 2 + ly[0] ** 2 + lz[0] ** 2)))
    w = rel_amp * rq / rl
    qx += w * lx; qy += w * ly; qz += w * lz
    return qx, qy, qz, w
