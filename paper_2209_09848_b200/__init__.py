"""B200-native matched-filter trajectory search (hot path of arXiv 2209.09848).

The product is the C-ABI library ``libtno_mf.so`` (CUDA, sm_100a; sources in ``csrc/``, interface
in ``include/tno_mf.h``).  This package is its thin Python binding plus a small convenience class.
"""
from .binding import (CAND_DTYPE, SOURCE_DTYPE, TRAJ_DTYPE, TnoMfError, make_sources,  # noqa: F401
                      tno_mf_background, tno_mf_best, tno_mf_create, tno_mf_debug_poison_shared, tno_mf_destroy, tno_mf_flux, tno_mf_inject, tno_mf_inject_ex, tno_mf_last_error,
                      tno_mf_last_kernel_ms, tno_mf_last_stats, tno_mf_local_z_static, tno_mf_last_work, tno_mf_peaks, tno_mf_plan, tno_mf_plan_slots,
                      tno_mf_search, tno_mf_search_ex, tno_mf_search_host, tno_mf_search_host_max, tno_mf_search_masked, tno_mf_search_max, tno_mf_set_prf_table, tno_mf_set_prf_table2d, tno_mf_downsample,
                      tno_mf_scatter_fit, tno_mf_scatter_lossgrad, tno_mf_scatter_subtract,
                      tno_mf_version)
from .search import MatchedFilter  # noqa: F401
