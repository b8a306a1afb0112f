"""Seeded synthetic inputs for the five BASELINE.json configs.

This package is DATA ONLY: it builds initial states (conserved variables on patches) and
the patch geometry tables.  It holds none of the solver's arithmetic (no slopes, no
Riemann solvers, no updates), imports neither ``oracle`` nor ``paper_1412_0934_b200``,
and its arrays are handed to both as plain numpy buffers.

Recipes: SURVEY.md §8(d) (configs 1-5, readings A15, A16, A21); restated in DESIGN.md §4.
"""
from .configs import (  # noqa: F401
    SEED,
    FIELDS_HYDRO,
    FIELDS_MHD,
    Level,
    Workload,
    morton_patch_origins,
    gaussian_random_field,
    solenoidal_random_field,
    primitive_to_conserved,
    split_into_patches,
    add_ghost_frame,
    strip_ghost_frame,
    config1_sod,
    config2_random_patches,
    config3_orszag_tang,
    config4_two_level,
    two_level_outflow,
    config_hierarchy,
    nested_hierarchy_from_fine,
    select_blocks,
    blocks_to_origins,
    origins_to_blocks,
    patch_flags_to_block_grid,
    config5_turbulence,
    smooth_wave_patchset,
    uniform_grid_workload,
    morton_permutation,
    turbulence_patches_torch,
    refined_level_cells,
)
