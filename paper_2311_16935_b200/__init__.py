"""B200-native hot path of the matrix-based omnidirectional pressure integration (arXiv 2311.16935).

The product is the C-ABI library libomni.so (include/omni.h, csrc/); this package is its thin ctypes binding.
Importing the package does not load the library; the first call does, and fails loudly when it is missing.
"""
from .binding import (Info, OmniError, SYMBOLS, apply_M, constants, launch_count, lib, profile_enable,  # noqa: F401
                      profile_read, release_memory, residual, set_loop_mode, solve, solve_batch2d, solve_cascade, solve_direct, source, status_string, velocity_source, version, workspace_bytes,
                      rans_source, compressible_rans_source, solve_guess, set_history, solve_pcg, solve_ex, Options, slab_plan, solve_slab, solve_slab_rank, slab_comm_create,
                      slab_comm_destroy, source_noalloc, source_noalloc_max_cells, resident_plan, resident_split)

# the C names, for callers who think in terms of include/omni.h
omni_solve = solve
omni_solve_batch2d = solve_batch2d
omni_solve_direct = solve_direct
omni_solve_guess = solve_guess
omni_solve_cascade = solve_cascade
omni_solve_pcg = solve_pcg
omni_solve_ex = solve_ex
omni_solve_slab = solve_slab
omni_slab_plan = slab_plan
omni_source = source
omni_velocity_source = velocity_source
omni_rans_source = rans_source
omni_compressible_rans_source = compressible_rans_source
omni_apply_M = apply_M
omni_residual = residual
omni_constants = constants
omni_workspace_bytes = workspace_bytes
omni_launch_count = launch_count
omni_set_loop_mode = set_loop_mode
omni_set_history = set_history
omni_release_memory = release_memory
omni_profile_enable = profile_enable
omni_profile_read = profile_read
omni_status_string = status_string
omni_version = version
