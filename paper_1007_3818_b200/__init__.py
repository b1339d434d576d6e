"""paper_1007_3818_b200 — B200-native hot path of GAMER's MUSCL-Hancock + Roe hydrodynamic solver
(arXiv 1007.3818): a C-ABI CUDA library (csrc/, include/gamer_hydro.h) and its thin binding."""
from .binding import (BC_OUTFLOW, BC_PERIODIC, MINMOD, PATH_AUTO, PATH_FUSED, PATH_FUSED_DUO, PATH_FUSED_SCALAR, PATH_GENERIC, VANLEER, MC, FLAG_ENTROPY_FIX, FLAG_HLLE_FALLBACK, GamerHydroError,  # noqa: F401
                      gamer_hydro_alloc, gamer_hydro_free, gamer_hydro_launch_count, gamer_hydro_set_path,
                      gamer_hydro_status, gamer_hydro_step, gamer_hydro_step_f64, gamer_hydro_step_host,
                      gamer_hydro_strerror, gamer_hydro_max_speed, gamer_hydro_fill_ghosts, gamer_hydro_advance, gamer_hydro_step_grid, gamer_hydro_set_guard_map, gamer_rtvd_step, gamer_hydro_step_ex, gamer_hydro_step_ex_f64,
                      gamer_hydro_max_speed_noalloc, gamer_hydro_max_speed_noalloc_limit, gamer_hydro_set_hlle_map)
