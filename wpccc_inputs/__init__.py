"""Seeded, synthetic input generators for the WP-CCC hot path.

This package builds the *inputs* both the CPU oracle (``oracle/``) and the CUDA
library consume: radial basis tables on the r-grid, trapezoid weights, impact
parameter sets and the five BASELINE.json workloads.  It contains none of the
method's arithmetic (no matrix elements, no quadrature of couplings, no
propagation) and imports neither ``oracle`` nor ``paper_2403_04252_b200``.
"""
from .basis import (Centre, Problem, make_centre, make_problem, hydrogenic_bound_u,
                    coulomb_wave_table, splitmix64_uniform, radial_grid)
from .configs import CONFIGS, build_config, log_spaced, tiny_problem

__all__ = ["Centre", "Problem", "make_centre", "make_problem", "hydrogenic_bound_u",
           "coulomb_wave_table", "splitmix64_uniform", "radial_grid", "CONFIGS",
           "build_config", "log_spaced", "tiny_problem"]
