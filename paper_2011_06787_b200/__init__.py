"""B200-native SPIIR hot path (arXiv 2011.06787): filter bank + coherent sky search.

The product is the C-ABI library ``libspiir_b200.so`` (include/spiir.h), hand-written
CUDA for sm_100a; this package is its thin ctypes binding.  PyTorch is used by the
callers for device memory and streams only.  Nothing here imports ``oracle``.
"""
from .binding import (  # noqa: F401
    lib, last_error, SpiirError, EXPORTS, LIB_PATH,
    spiir_bank_desc, spiir_snr_view, spiir_band_plan, TRIGGER_DTYPE, RESULT_DTYPE,
    make_desc, Bank, SkyPlan, SkyPlanSet, SnrView, sky_table_build, sky_table_set_build, sky_table_nearest, upsample_windows,
    triggers_to_numpy, triggers_from_numpy, results_to_numpy,
    XI2_DTYPE, template_autocorr, signal_consistency, xi2_to_numpy,
    RANK_DTYPE, spiir_rank_bins, Ranker, rank_to_numpy, rank_static, SPIIR_RANK_STATIC_MAX_BINS, spiir_frontend_desc, FrontEnd,
    SPIIR_OK, SPIIR_EINVAL, SPIIR_ENOMEM, SPIIR_ECUDA, SPIIR_EOVERFLOW,
)
from . import binding as _b

for _n in EXPORTS:                      # the C names themselves: spiir_bank_init, spiir_filter_chunk, ...
    globals()[_n] = getattr(_b, _n)
