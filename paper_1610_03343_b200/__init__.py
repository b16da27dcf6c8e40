"""B200-native write-conflict-free many-body force evaluation (arXiv 1610.03343 hot path).

Python names mirror the C ABI of include/md.h one to one; see `binding.py`.
"""
from .binding import *  # noqa: F401,F403
from .binding import (EXPORTS, MDError, Neighbors, lib_path, load, md_build_neighbors, md_neighbors_create,
                      md_neighbors_destroy, md_neighbors_export, md_neighbors_import, md_neighbors_status,
                      md_npt_run, md_nve_heat_run, md_nve_run, md_nve_run_host, md_pair_counts, md_probe_fp64_peak, md_profile_enable, md_profile_read, md_sw_force, md_tersoff_force, md_tersoff_force_literal, md_tersoff_multi_force,
                      md_velocity_verlet_step, md_version)
