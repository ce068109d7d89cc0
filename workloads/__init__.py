"""Seeded synthetic inputs shared by the oracle tests and the CUDA library tests/bench.

This package holds NO arithmetic of the method (no reference elements, no DG operators, no HABC
coefficients): only meshes, material tables, closed-form initial fields and the named configurations
of BASELINE.json.  Both `oracle/` and `paper_1610_05023_b200/` consume its outputs; neither of them
imports the other.
"""
from .configs import (CONFIGS, Workload, cube_mesh, layered_speed, initial_fields, make_workload,
                      scaled_workload)

__all__ = ["CONFIGS", "Workload", "cube_mesh", "layered_speed", "initial_fields", "make_workload",
           "scaled_workload"]
