"""Seeded synthetic inputs shared by the oracle tests and the CUDA path.

This module holds *only* input generation (random numbers, particle clouds,
force vectors, random-init MLP weights).  None of the method's arithmetic
(MLP evaluation, tree, admissibility, ACA, mat-vec) lives here, so that the
oracle (`oracle/`) and the product (`paper_2505_08174_b200/`) share no code.

Recipes follow SURVEY.md §8(d) / DESIGN.md "Input recipe".
"""
from .rng import splitmix64, uniform01, normal01  # noqa: F401
from .generators import (  # noqa: F401
    cube_cloud, ball_cloud, chain_cloud, lattice_cloud, line_points, lattice_drop, two_drops, filament_sphere, mixture_forces,
    gaussian_forces, gravity_forces, filament_forces,
    xavier_mlp, MLP2_DIMS, MLP3_DIMS, MLP2_PAPER_DIMS, config, CONFIGS,
)
