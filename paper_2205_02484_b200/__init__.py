"""paper_2205_02484_b200 — B200-native (sm_100a) HARM update of ideal GR-MHD (cuHARM, arXiv 2205.02484).

A thin ctypes binding of libcuharm.so (include/cuharm.h): argument marshalling only — every step of the
path runs in the library's CUDA kernels.  PyTorch supplies device memory and the stream; nothing else.
There is no CPU path: on a machine without the built library or without a CUDA device the calls raise.
"""
from .binding import (CuharmError, CuharmParams, Solver, lib, make_params, lib_path,  # noqa: F401
                      cuharm_grid_init, cuharm_workspace_bytes, cuharm_bind, cuharm_metric_precompute,
                      cuharm_step, cuharm_step_cfl, cuharm_get_time, cuharm_apply_floors, cuharm_cons_to_prim, cuharm_prim_to_cons, cuharm_cfl_dt, cuharm_last_cfl_dt,
                      cuharm_divb, cuharm_divb_noalloc, cuharm_shell_fluxes, cuharm_get_geom, cuharm_apply_bc, cuharm_flux_dir, cuharm_get_stats,
                      cuharm_use_graph, cuharm_launch_count, cuharm_set_timing, cuharm_get_timing, KERNEL_CLASSES, cuharm_destroy, cuharm_strerror)
