"""B200-native orbit-library construction (the hot path of arXiv 2607.00117 fixed by BASELINE.json).

The product is libschwarmax.so (hand-written CUDA for sm_100a behind the C ABI of include/schwarmax.h);
this package holds its sources (csrc/), the build step, a thin ctypes binding and the seeded inputs.
"""
from . import inputs  # noqa: F401
from .binding import (SchwarmaxError, sm_build_bundled_library, sm_build_gh_library, sm_build_library, sm_build_observable_library, sm_build_observable_library_batch, sm_build_library_batch, sm_eval_force, sm_flush_rows, sm_stage_library_batch, sm_stage_library_noalloc,  # noqa: F401
                      sm_free_potential, sm_integrate_trajectories, sm_last_kernel_times, sm_launch_count, sm_make_potential,
                      sm_make_potential_batch, sm_measure_fma_peak, sm_set_debug_flags, sm_solve_weights, sm_marginal_chi2, sm_last_solve_times, sm_version)
