"""Seeded synthetic inputs shared by the oracle tests and the CUDA path.

This module holds NONE of the method's arithmetic (no interpolation, no ODE
stepping, no Q formula, no Sobel, no refinement).  It only manufactures
*data*: magnetic-field cubes sampled from analytic formulas, seed arrays and
the five benchmark configurations of BASELINE.json.  Both `oracle/` (through
the tests) and `paper_1609_00724_b200` (through tests and bench.py) consume
the arrays produced here; neither implementation imports the other.

The paper's own datasets (Titov-Demoulin flux rope; the
SOL2010-04-08 NLFFF model) are not available; the synthetic
configurations D1..D5 stand
in for them.
"""
from .rng import SplitMix64
from .fields import (
    Grid,
    uniform_field,
    hyperbolic_field,
    hyperbolic_B,
    quadrupole_charges,
    quadrupole_B,
    quadrupole_field,
    lfff_modes,
    lfff_B,
    lfff_field,
    superposition_field,
    stretched_axis,
)
from .seeds import lattice_seeds, Lattice
from .configs import make_config, CONFIG_NAMES

__all__ = [
    "SplitMix64", "Grid", "uniform_field", "hyperbolic_field", "hyperbolic_B",
    "quadrupole_charges", "quadrupole_B", "quadrupole_field", "lfff_modes",
    "lfff_B", "lfff_field", "superposition_field", "stretched_axis",
    "lattice_seeds", "Lattice", "make_config", "CONFIG_NAMES",
]
