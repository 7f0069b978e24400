"""Seed lattices (data only).  Seeds are pixel-centred (reading A14): the seed lattice is independent
of the field grid; arbitrary planar slices are just a choice of origin and edge vectors."""
from __future__ import annotations

import dataclasses

import numpy as np


@dataclasses.dataclass
class Lattice:
    """Level-0 seed lattice: seed(c) = origin + sum_d (c_d + 0.5)/n_d * e_d, c_d in [0, n_d)."""
    ndim: int
    n: tuple          # (n0, n1, n2); n2 = 1 for 2-D
    origin: tuple
    e0: tuple
    e1: tuple
    e2: tuple = (0.0, 0.0, 0.0)

    @property
    def count(self):
        return int(self.n[0]) * int(self.n[1]) * int(self.n[2])


def lattice_seeds(lat: Lattice) -> np.ndarray:
    """Level-0 seeds in dense index order (c2*n1 + c1)*n0 + c0, shape (count, 3), fp64."""
    n0, n1, n2 = (int(v) for v in lat.n)
    w0 = (np.arange(n0, dtype=np.float64) + 0.5) / n0
    w1 = (np.arange(n1, dtype=np.float64) + 0.5) / n1
    w2 = (np.arange(n2, dtype=np.float64) + 0.5) / n2 if lat.ndim == 3 else np.zeros(1)
    o = np.asarray(lat.origin, dtype=np.float64)
    e0 = np.asarray(lat.e0, dtype=np.float64); e1 = np.asarray(lat.e1, dtype=np.float64)
    e2 = np.asarray(lat.e2, dtype=np.float64)
    out = np.empty((n2, n1, n0, 3), dtype=np.float64)
    for k in range(3):
        out[..., k] = o[k] + w0[None, None, :] * e0[k] + w1[None, :, None] * e1[k] + w2[:, None, None] * e2[k]
    return out.reshape(-1, 3)
