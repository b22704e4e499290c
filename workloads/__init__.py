"""Seeded synthetic input generators shared by the oracle and the CUDA path.

This package holds NONE of the method's arithmetic (no sweep, no moments, no
boundary-condition evaluation): it only builds plain numpy arrays -- grids,
masks, band tables, quadrature tables, heat-source fields, boundary-condition
codes -- that are handed verbatim to `oracle/` and to the C-ABI CUDA library.
It imports neither of them.

Recipes follow SURVEY.md section 8(d) / BASELINE.json `configs[0..4]`; they
stand in for the paper's workloads (silicon films and FinFET meshes,
PAPER.md:48, 58, 96, 106) whose meshes and DFT band tables are not available.
"""
from .configs import (  # noqa: F401
    BC_ISOTHERMAL, BC_DIFFUSE, BC_SPECULAR, BC_PERIODIC,
    FP64, FP32_STORE_FP64_ACC,
    Problem, band_table, quadrature_3d, quadrature_1d, quadrature_gl_theta_octant,
    config, CONFIG_NAMES, MASTER_SEED, random_problem,
)
