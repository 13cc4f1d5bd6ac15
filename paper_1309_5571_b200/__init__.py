"""B200-native (sm_100a, FP64) DMRG hot path of arXiv:1309.5571: the sector-blocked superblock
projection  X'_jl += A_{i->j} X_ik B_{k->l}^T as grouped DMMA launches and the
Davidson BLAS-2 kernels as HBM streams, behind the C ABI of include/dmrg_b200.h.

This package is the thin Python binding (argument marshalling only).  It never imports `oracle/`.
"""
from .binding import (Plan, DmrgError, Stats, load_library, LIB_PATH, EXPORTS,
                      dmrg_plan_create, dmrg_apply_H, dmrg_davidson_step, dmrg_lowest_eigenpair,
                      dmrg_probe_fp64_peak, dmrg_probe_hbm_read, sector_eig, select_states, infinite_heisenberg, gemv_trans_static,
                      DMRG_OK, DMRG_NOT_CONVERGED, DMRG_E_INVALID_ARG, DMRG_E_SECTOR, DMRG_E_ALLOC,
                      DMRG_E_CUDA, DMRG_E_NUMERIC, DMRG_HEISENBERG, DMRG_HUBBARD)

__all__ = ["Plan", "DmrgError", "Stats", "load_library", "LIB_PATH", "EXPORTS", "dmrg_plan_create",
           "dmrg_apply_H", "dmrg_davidson_step", "dmrg_lowest_eigenpair", "dmrg_probe_fp64_peak",
           "dmrg_probe_hbm_read", "sector_eig", "select_states", "infinite_heisenberg", "gemv_trans_static"]
