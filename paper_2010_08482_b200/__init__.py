"""B200-native CT-HYB local-trace library (arXiv:2010.08482, Eq. 65): Python face of libctqmc_b200.so.

Everything here is argument marshalling around the C ABI of include/ctqmc.h; the names are the C names.
"""
from . import binding  # noqa: F401
from .binding import (  # noqa: F401
    CTQMC_OPT_PANEL_WIDTH, CTQMC_OPT_PATH, CTQMC_OPT_SCHEDULE, CTQMC_OPT_SCRATCH_LIMIT, CTQMC_PATH_AUTO, CTQMC_PATH_GROUPED, CTQMC_PATH_LARGE, CTQMC_PATH_PANEL, CTQMC_PATH_SMALL, CTQMC_OPT_TIMING, CTQMC_SCHEDULE_LITERAL, CTQMC_SCHEDULE_THIN, CTQMC_STATUS_INVALID,
    CTQMC_STATUS_OK, CTQMC_STATUS_VANISHING, CtqmcError, EXPORTS, ImpurityHandle, LIB_PATH, ctqmc_bound_batch,
    ctqmc_bound_batch_host, ctqmc_free_impurity, ctqmc_last_error, ctqmc_last_stats, ctqmc_last_timing, ctqmc_load_impurity, ctqmc_measure_fp64_peak,
    ctqmc_set_option, ctqmc_trace_batch, ctqmc_trace_batch_host, library,
)
