"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NO arithmetic of the method (no Fourier sums, no response
functions, no binning): it only builds real-space samples, detector grids and
rotation matrices as NumPy arrays.  Both `oracle/` and the CUDA binding consume
the arrays produced here; neither imports the other.

Recipes follow SURVEY.md Appendix C (configs C1..C5 of BASELINE.json) and are
restated in DESIGN.md.
"""
from .samples import (  # noqa: F401
    rot_y, rot_z, rotation_alpha_beta,
    sphere_node_centred, sphere_cell_centred,
    Workload, KINDS, KIND_INDEX, ALL_KINDS,
    polar_grid, cartesian_grid, list_grid,
    config_c1, config_c2, config_c3, config_c4, config_c5, config_fig10, make_config,
    q_subset, uniform_sphere_sample, linear_vortex_sphere_sample, cuboid_lattice,
)
