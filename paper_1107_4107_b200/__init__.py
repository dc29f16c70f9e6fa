"""paper_1107_4107_b200 — B200-native (sm_100a) hot path of arXiv 1107.4107: ensemble symplectic
integration of the paper's 3-d.o.f. Hamiltonian -> Arnold-web maps (FLI image + visited-cell density).

The product is libaw.so (hand-written CUDA behind the C ABI of include/aw.h).  This package is the
thin Python binding: argument marshalling only.  PyTorch is used for device memory and streams.
There is no CPU fallback: importing the binding without the built library raises.
"""
from .binding import (AW_DENS_ACTION, AW_DENS_VEL_BOTH, AW_DENS_VEL_LOWER, AW_DENS_VEL_UPPER,
                      AW_IND_CLASS, AW_IND_DH, AW_IND_DHS, AW_IND_DP, AW_IND_FLI, AW_IND_FTLE, AW_IND_VX, AW_IND_VY,
                      AW_IND_VZ, AW_SHAPE_DISK, AW_SHAPE_GAUSS, AW_SHAPE_GRID, AW_SHAPE_RECT, AW_SHAPE_SPHERE,
                      AW_ST_LEFT, AW_ST_LIVE, AW_ST_NONFINITE, AW_ST_OFFSHELL, AW_ST_RANGE, AwError, Ensemble, Grid,
                      aw_block_size, aw_bound_energy, aw_common_tangent, aw_density, aw_energy_stats, aw_energy_stats_noalloc,
                      aw_energy_stats_scratch_bytes, AW_NOALLOC_MAX_N,
                      aw_indicator, aw_init_shell, aw_integrate, aw_kernel_schedule, aw_launch_count, aw_map_host, aw_mark, aw_velocity_map_host,
                      aw_stage_constants, aw_state_bytes, aw_strerror, aw_trig_level, aw_version, lib, make_grid)
from .configs import CONFIGS

__all__ = [n for n in dir() if n.startswith(("aw_", "AW_")) or n in
           ("AwError", "Ensemble", "Grid", "lib", "make_grid", "CONFIGS")]
