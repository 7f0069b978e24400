"""The five synthetic workloads of BASELINE.json `configs`, as data.

`make_config(name, scale)` returns a dict of plain numpy arrays / numbers.  `scale` < 1 shrinks the field
grid and the seed lattice by that factor per axis (parity-test sizes the oracle finishes in seconds);
scale = 1 is the full size bench.py times.
"""
from __future__ import annotations

import math

import numpy as np

from .fields import (Grid, hyperbolic_field, quadrupole_charges, quadrupole_B, quadrupole_field, lfff_modes,
                     lfff_field, superposition_field)
from .seeds import Lattice, lattice_seeds

CONFIG_NAMES = ("cfg1", "cfg2", "cfg3", "cfg4", "cfg5")

TRACE_L, TRACE_LQ = 0, 1


def _sc(n, scale, lo=4):
    return max(lo, int(round(n * scale)))


def _max_steps(grid: Grid, step_frac: float) -> int:
    return int(8 * (grid.nx + grid.ny + grid.nz) / step_frac)


def make_config(name: str, scale: float = 1.0, with_seeds: bool = True) -> dict:
    if name == "cfg1":
        # BASELINE.json configs[0]: hyperbolic k=2, fp64 64^3 on [-1,1]^2 x [0,1]; 128x128 seeds on z=0 in [-0.5,0.5]^2
        g = Grid.uniform((_sc(64, scale),) * 3, (-1, -1, 0), (1, 1, 1))
        B = hyperbolic_field(g, 2.0)
        ns = _sc(128, scale)
        lat = Lattice(2, (ns, ns, 1), (-0.5, -0.5, 0.0), (1.0, 0, 0), (0, 1.0, 0))
        cfg = dict(grid=g, B=B, sample_type="f64", lattice=lat, mode=TRACE_LQ, levels=0, k=2.0)
    elif name in ("cfg2", "cfg3"):
        # configs[1], [2]: quadrupole of 4 charges at depth 0.1, fp64 128^3 on [-1,1]^2 x [0,1]
        g = Grid.uniform((_sc(128, scale),) * 3, (-1, -1, 0), (1, 1, 1))
        q, r = quadrupole_charges()
        B = quadrupole_field(g, q, r)
        if name == "cfg2":
            ns = _sc(1024, scale)
            lat = Lattice(2, (ns, ns, 1), (-0.6, -0.6, 0.0), (1.2, 0, 0), (0, 1.2, 0))
            cfg = dict(grid=g, B=B, sample_type="f64", lattice=lat, mode=TRACE_LQ, levels=0, charges=(q, r),
                       bz_min=1e-3)
        else:
            n0, n1 = _sc(2048, scale), _sc(1024, scale)
            lat = Lattice(2, (n0, n1, 1), (-0.6, 0.0, 0.0), (1.2, 0, 0), (0, 0, 0.5))
            cfg = dict(grid=g, B=B, sample_type="f64", lattice=lat, mode=TRACE_L, levels=4, p=0.95, charges=(q, r))
    elif name == "cfg4":
        # configs[3]: LFFF alpha=1.5, 32 modes, fp32 samples 256^3 on [0,1]^3, 256^3 seeds at cell centres
        n = _sc(256, scale)
        g = Grid.uniform((n, n, n), (0, 0, 0), (1, 1, 1))
        modes = lfff_modes()
        B = lfff_field(g, modes)
        lat = Lattice(3, (n, n, n), (0.0, 0.0, 0.0), (1.0, 0, 0), (0, 1.0, 0), (0, 0, 1.0))
        cfg = dict(grid=g, B=B, sample_type="f32", lattice=lat, mode=TRACE_LQ, levels=0, modes=modes)
    elif name == "cfg5":
        # configs[4]: quadrupole (shifted by +0.5,+0.5) + w*LFFF, fp32 samples 512x512x256 on [0,1]^2 x [0,0.5]
        nx, nz = _sc(512, scale), _sc(256, scale)
        g = Grid.uniform((nx, nx, nz), (0, 0, 0), (1, 1, 0.5))
        q, r = quadrupole_charges(shift=(0.5, 0.5))
        modes = lfff_modes()
        bx, by, bz, w = superposition_field(g, q, r, modes, 0.1)
        lat = Lattice(3, (nx, nx, nz), (0.0, 0.0, 0.0), (1.0, 0, 0), (0, 1.0, 0), (0, 0, 0.5))
        cfg = dict(grid=g, B=(bx, by, bz), sample_type="f32", lattice=lat, mode=TRACE_L, levels=3, p=0.95,
                   charges=(q, r), modes=modes, lfff_weight=w)
    else:
        raise ValueError(f"unknown config {name!r}")

    g = cfg["grid"]
    cfg["name"] = name
    cfg["scale"] = scale
    cfg["box_lo"] = tuple(g.lo)
    cfg["box_hi"] = tuple(g.hi)
    cfg["step_frac"] = 0.25
    cfg["max_steps"] = _max_steps(g, 0.25)
    cfg["null_eps"] = 1e-12
    cfg["max_length"] = math.inf
    if with_seeds:
        seeds = lattice_seeds(cfg["lattice"])
        if name == "cfg2":
            q, r = cfg["charges"]
            keep = np.abs(quadrupole_B(seeds, q, r)[:, 2]) > cfg["bz_min"]
            cfg["keep"] = keep
            seeds = np.ascontiguousarray(seeds[keep])
        cfg["seeds"] = seeds
    return cfg
