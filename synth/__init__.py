"""Seeded synthetic inputs shared by the oracle and the CUDA path.

This package holds NONE of the method's arithmetic (no field, torque, FFT, tensor or
Runge-Kutta code): only a counter-based random generator, the parameter container and the
recipes that build the BASELINE.json configurations C1..C5.
Both `oracle/` and `paper_1406_7635_b200/` are fed the arrays made here; neither imports
the other.
"""
from .rng import hash64, uniform01, random_unit_vectors
from .params import Params
from .configs import (SEED0, config_c1, config_c2, config_c3, config_c4, config_c4_regions,
                      config_c5, voronoi_regions)

__all__ = ["hash64", "uniform01", "random_unit_vectors", "Params", "SEED0", "config_c1",
           "config_c2", "config_c3", "config_c4", "config_c4_regions", "config_c5", "voronoi_regions"]
