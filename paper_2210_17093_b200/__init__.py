"""B200-native qsGW correlation self-energy build (arxiv 2210.17093, Eqs. (17)-(19), RI form).

The product is the C-ABI library ``libqsgw_sigma.so`` (include/qsgw_sigma.h; sources in csrc/).
This package is its thin Python binding: same names, argument marshalling only.
"""
from .binding import (  # noqa: F401
    LIB_PATH, EXPORTS, Plan, QsgwSigmaError, load_library,
    qsgw_sigma_create, qsgw_sigma_build, qsgw_sigma_begin, qsgw_sigma_add_poles, qsgw_sigma_finish,
    qsgw_sigma_build_host, qsgw_sigma_diag_build, qsgw_mp2_direct_build, qsgw_mp2_build, qsgw_ri_ao_to_mo, qsgw_ri_ao_to_mo_work_doubles, qsgw_ri_ao_to_mo_static, qsgw_ri_ao_to_mo_static_max_doubles,
    qsgw_sigma_destroy, qsgw_sigma_last_error, qsgw_sigma_workspace_bytes,
    qsgw_sigma_limit_pole_batch, qsgw_sigma_set_profiling, qsgw_sigma_get_stats, qsgw_sigma_set_debug, qsgw_sigma_version, qsgw_sigma_pole_slice,
    qsgw_casida_work_doubles, qsgw_casida_matrix, qsgw_casida_z,
    QSGW_SIGMA_OK, QSGW_SIGMA_ERR_INVALID_ARG, QSGW_SIGMA_ERR_ALLOC, QSGW_SIGMA_ERR_CUDA,
)
from .sharded import allreduce_sigma, qsgw_sigma_build_pole_sharded  # noqa: F401,E402
