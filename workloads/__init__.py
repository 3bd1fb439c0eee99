"""Seeded synthetic input generators shared by the oracle tests and the CUDA path.

This package holds none of the arithmetic of the method under test (no particle-particle
sum, no predictor): it only draws Plummer-sphere initial conditions and the derivative
values the predictor will later consume (those come from the closed-form derivatives of
one smooth analytic field; generator data, never an expected value).  See DESIGN.md "Input recipe".
"""
from .plummer import (CONFIGS, Workload, make_workload, make_config, lattice_workload,
                      splitmix64_uniform, A_PLUMMER)

__all__ = ["CONFIGS", "Workload", "make_workload", "make_config", "lattice_workload",
           "splitmix64_uniform", "A_PLUMMER"]
