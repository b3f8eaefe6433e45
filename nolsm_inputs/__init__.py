"""Seeded synthetic input generators shared by the oracle, the tests and bench.py.

This package holds *inputs only*: positions, block-sparse H and S, microbench matrices.
It contains none of the NOLSM method's arithmetic (no inverse, no sign function, no density
matrix, no chemical-potential search) and imports neither ``oracle`` nor the CUDA package.
The recipe is the one stated in BASELINE.json:configs and completed in DESIGN.md ("Input recipe").
"""
from .rng import splitmix64, uniform_u53
from .water import (GRID_PER_ANGSTROM, BS, N_OCC_PER_MOL, N_ELEC_PER_MOL, WaterSystem,
                    make_positions, make_water_system, model_parameters, CONFIGS)
from .dense import make_gapped_symmetric, microbench_batch

__all__ = [
    "splitmix64", "uniform_u53", "GRID_PER_ANGSTROM", "BS", "N_OCC_PER_MOL", "N_ELEC_PER_MOL",
    "WaterSystem", "make_positions", "make_water_system", "model_parameters", "CONFIGS", "make_gapped_symmetric",
    "microbench_batch",
]
