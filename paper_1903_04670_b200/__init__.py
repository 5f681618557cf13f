"""B200-native multi-species DGFS Boltzmann collision operator (arXiv 1903.04670).

Thin Python binding over the C-ABI library `libdgfs.so` (include/dgfs.h).  Argument marshalling
only: every step of the path runs in the library's CUDA kernels.  PyTorch provides device memory
and streams.  There is no CPU fallback: importing works anywhere (so the ABI can be inspected),
but creating a context without the built library or without a CUDA device raises.
"""
from .api import (DgfsError, Dgfs, Mesh1D, load_library, library_path, exported_symbols,
                  dgfs_create, dgfs_collide, dgfs_collide_pairs, dgfs_step, dgfs_step_euler, dgfs_advect_rhs,
                  dgfs_destroy, dgfs_reserve, dgfs_workspace_bytes, dgfs_get_quadrature,
                  dgfs_get_tables, dgfs_flops_per_pair_eval, dgfs_last_error,
                  dgfs_launch_count, dgfs_profile_enable, dgfs_profile_count, dgfs_profile_get,
                  dgfs_profile_reset, dgfs_collide_host, dgfs_measure_fp64_peak, dgfs_table_bytes, dgfs_measure_dft,
                  dgfs_collide_noalloc, dgfs_measure_fp64_mix)
from . import api

__all__ = [
    "DgfsError", "Dgfs", "Mesh1D", "load_library", "library_path", "exported_symbols",
    "dgfs_create", "dgfs_collide", "dgfs_collide_pairs", "dgfs_step", "dgfs_step_euler", "dgfs_advect_rhs",
    "dgfs_destroy", "dgfs_reserve", "dgfs_workspace_bytes", "dgfs_get_quadrature",
    "dgfs_get_tables", "dgfs_flops_per_pair_eval", "dgfs_last_error",
    "dgfs_launch_count", "dgfs_profile_enable", "dgfs_profile_count", "dgfs_profile_get",
    "dgfs_profile_reset", "dgfs_collide_host", "dgfs_measure_fp64_peak", "dgfs_table_bytes", "dgfs_measure_dft", "dgfs_collide_noalloc", "dgfs_measure_fp64_mix", "api",
]
