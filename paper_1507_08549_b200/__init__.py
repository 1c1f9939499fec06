"""B200-native self-gravity Poisson solve of arXiv 1507.08549 (multipole boundary + red-black SOR, fp64).

The product is the C-ABI library ``libsn_poisson.so`` (include/sn_poisson.h); this package is its thin binding.
"""
from .binding import (EXPORTS, EXPORTS_LEVELSET, EXPORTS_WENO, sn_weno_create, sn_weno_destroy, sn_weno_evolve,
                      sn_weno_get_stat, sn_weno_last_error, sn_weno_max_speeds, sn_weno_rhs, sn_weno_rhs_host, sn_weno_step, sn_levelset_create, sn_levelset_destroy, sn_levelset_get_stat,
                      sn_levelset_last_error, sn_levelset_reinit, sn_levelset_reinit_host, LIB_PATH, SnPoissonError, load, sn_poisson_create, sn_poisson_destroy,
                      sn_poisson_get_boundary, sn_poisson_get_history, sn_poisson_get_moments,
                      sn_poisson_get_omega, sn_poisson_get_stat, sn_poisson_moments_static, sn_poisson_gravity, sn_poisson_last_error,
                      sn_poisson_result,
                      sn_poisson_set_boundary, sn_poisson_set_omega, sn_poisson_set_stop_rule, sn_poisson_solve_gravity, sn_poisson_solve_mg, sn_poisson_solve_mg_batch, sn_poisson_solve_mg_batch_host, sn_poisson_solve_mg_host, sn_poisson_set_option, sn_poisson_solve,
                      sn_poisson_solve_batch, sn_poisson_solve_batch_host, sn_poisson_solve_host,
                      sn_poisson_solve_sequence_host, sn_poisson_probe_l2, sn_poisson_version)
from .solver import LevelSet, PoissonSolver, Weno

__all__ = ["PoissonSolver", "LevelSet", "Weno", "SnPoissonError", "EXPORTS", "LIB_PATH", "load", "sn_poisson_result"] + list(EXPORTS) + list(EXPORTS_LEVELSET) + list(EXPORTS_WENO)
