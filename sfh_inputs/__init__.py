"""Seeded synthetic inputs (meshes and initial conditions) for the five BASELINE.json configs.

This module serves BOTH the CPU oracle and the CUDA path and therefore holds none of the
method's arithmetic (no fluxes, no limiter, no prolongation/restriction, no CFL): it only
produces octree block lists and pointwise-evaluated initial fields.  Recipes are stated in
DESIGN.md ("Synthetic inputs").  Arrays: U[b][v][k][j][i], v = (rho, rho vx, rho vy, rho vz,
rho E) with rho E = P/(gamma-1) + rho |v|^2 / 2 (eq. 8); ijk[b] = (bx, by, bz).
"""
from .mesh import Tree, uniform_tree, tree_from_criterion, blockify, unblockify  # noqa: F401
from .fields import (gaussian_random_field, lognormal_density, velocity_field, hash_normal,  # noqa: F401
                     prim_to_cons)
from .configs import make_config, CONFIG_NAMES, Problem  # noqa: F401
from .small import small_amr_tree, smooth_fields, problem_from_tree, add_scalars  # noqa: F401
from .blocks16 import to16, tree16_problem, split_state, merge_state, split_blocks  # noqa: F401
