"""Seeded synthetic inputs for the five BASELINE.json configs.

This module is DATA ONLY.  It is the one piece shared by the CPU oracle
(`oracle/`) and the CUDA path (`paper_2305_13555_b200/`): it draws the random
numbers, lays out the arrays and names the boundary conditions.  It holds none
of the method's arithmetic (no quadrature, no matrices, no iteration) and
imports neither side.
"""
from .configs import Problem, make_problem, make_multi_region, CONFIG_NAMES, BC_VACUUM, BC_INCIDENT_ISOTROPIC, BC_REFLECTING  # noqa: F401
