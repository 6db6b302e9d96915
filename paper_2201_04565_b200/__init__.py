"""B200-native lattice-spring-model step (hot path of CuLSM, arXiv 2201.04565) behind a C ABI.

The product is liblsm_b200.so (include/lsm.h): hand-written CUDA kernels for sm_100a plus a C++ host runtime.
This package is the thin Python binding: argument marshalling only.  There is no CPU fallback: importing works
anywhere (so the symbol table can be checked), but creating a simulation without a CUDA device raises LsmError.
"""
from .binding import (  # noqa: F401
    LsmError, LsmSim, lsm_create, lsm_set_boundary, lsm_step, lsm_write_state, lsm_read_state, lsm_read_forces,
    lsm_read_broken, lsm_read_energy, lsm_read_virial, lsm_read_strain, lsm_read_stress, lsm_run_to_failure, lsm_set_strain_rate, lsm_compact, lsm_sync, lsm_get_info, lsm_destroy,
    lsm_last_error, lsm_abi_version, lsm_spring_energy_static, STATIC_MAX_SPRINGS, library, library_path, EXPORTS,
    FIXED, MOVE, FORCE_AUTO, FORCE_SCATTER, FORCE_GATHER, FORCE_SCATTER_WARP, FORCE_SCATTER_TILE, REORDER_NONE, REORDER_MORTON, REORDER_RCM, REORDER_BLOCKED, GATHER_AUTO, GATHER_DIRECT, GATHER_STREAMED, WINDOW_AUTO, WINDOW_ON, WINDOW_OFF, FUSION_AUTO, FUSION_ON, FUSION_OFF, FUSION_RESIDENT,
)
