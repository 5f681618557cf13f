"""Seeded synthetic workloads (configs c0..c4 of BASELINE.json / SURVEY.md section 8(d)).

This module serves BOTH the CPU oracle's tests and the CUDA path's tests/bench.  It holds
none of the method's arithmetic (no quadrature, no tables, no FFT, no collision operator):
only the velocity grid, Maxwellians and a counter-based random number generator.  The recipe
is written out in DESIGN.md ("Input recipe").
"""
from .rng import splitmix64_uniform
from .configs import CONFIGS, Config, get_config
from .inputs import velocity_nodes, maxwellian, make_points, make_dg_state

__all__ = [
    "splitmix64_uniform", "CONFIGS", "Config", "get_config",
    "velocity_nodes", "maxwellian", "make_points", "make_dg_state",
]
