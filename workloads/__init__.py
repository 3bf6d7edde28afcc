"""Seeded synthetic input generators shared by the oracle tests and the CUDA path.

This package holds NONE of the method's arithmetic (no radial basis, no moments,
no contraction): only lattices, perturbations, species draws, coefficient draws,
neighbour lists and the active-set matrix.  Recipe: DESIGN.md "Input recipe",
following BASELINE.json `configs` and SURVEY.md section 8(d).
"""
from .lattice import (CONFIGS, Workload, make_workload, neighbor_list_stencil,
                      neighbor_list_bruteforce, reverse_index, active_set_inverse,
                      random_cluster)

__all__ = ["CONFIGS", "Workload", "make_workload", "neighbor_list_stencil",
           "neighbor_list_bruteforce", "reverse_index", "active_set_inverse",
           "random_cluster"]
