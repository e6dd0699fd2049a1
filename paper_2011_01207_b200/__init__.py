"""paper_2011_01207_b200 -- thin Python binding of libtkhp (include/tkhp.h).

Real-space AMOEBA polarization (blocked neighbour list -> permanent field ->
T.mu / PCG solve -> energy) on one NVIDIA B200, after arXiv 2011.01207.

Argument marshalling only: every step of the path runs in the CUDA kernels of
``csrc/``.  PyTorch supplies device memory and streams, nothing else.  There is
no CPU fallback: importing works without a GPU (so the build can be checked),
but creating a context without a CUDA device raises, and a missing
``libtkhp.so`` raises at import of :mod:`paper_2011_01207_b200.binding`.
"""
from .binding import (TKHP_FP64, TKHP_MIXED, TKHP_FIXED, TKHP_LIST_TILES, TKHP_LIST_CLUSTER, TKHP_LIST_ATOM,
                      TKHP_SOLVER_NO_PERSISTENT, TKHP_SOLVER_NO_FUSED_STEP, TKHP_SOLVER_STORED_T,
                      TKHP_SOLVER_TEST_BARRIER_FAULT,
                      TkhpError, TkhpParams, Polarizer, lib, lib_path,
                      tkhp_workspace_bytes, tkhp_create, tkhp_destroy, tkhp_last_error,
                      tkhp_nblist_build, tkhp_nblist_view, tkhp_nblist_stats, tkhp_nblist_atom_stats,
                      tkhp_perm_field, tkhp_tmatvec, tkhp_polar_solve,
                      tkhp_polar_energy, tkhp_polar_energy_static, TKHP_STATIC_MAX_ATOMS,
                      tkhp_polarize_host, tkhp_last_timings,
                      tkhp_fma_peak, tkhp_profile_reset, tkhp_profile_read, tkhp_profile_read_solve, tkhp_profile_read_build,
                      EXPORTED_SYMBOLS)

__all__ = [
    "TKHP_FP64", "TKHP_MIXED", "TKHP_FIXED", "TKHP_LIST_TILES", "TKHP_LIST_CLUSTER", "TKHP_LIST_ATOM", "TKHP_SOLVER_NO_PERSISTENT", "TKHP_SOLVER_NO_FUSED_STEP", "TKHP_SOLVER_STORED_T", "TKHP_SOLVER_TEST_BARRIER_FAULT", "TkhpError",
    "TkhpParams", "Polarizer", "lib", "lib_path", "tkhp_workspace_bytes", "tkhp_create",
    "tkhp_destroy", "tkhp_last_error", "tkhp_nblist_build", "tkhp_nblist_view",
    "tkhp_nblist_stats", "tkhp_nblist_atom_stats", "tkhp_perm_field", "tkhp_tmatvec", "tkhp_polar_solve",
    "tkhp_polar_energy", "tkhp_polar_energy_static", "TKHP_STATIC_MAX_ATOMS", "tkhp_polarize_host", "tkhp_last_timings", "tkhp_fma_peak",
    "tkhp_profile_reset", "tkhp_profile_read", "tkhp_profile_read_solve", "tkhp_profile_read_build", "EXPORTED_SYMBOLS",
]
