"""Seeded synthetic inputs for the five BASELINE.json configurations.

This package is the ONLY thing the float64 oracle (``oracle/``) and the CUDA
path (``paper_2011_06787_b200/``) share.  It produces inputs — strain, filter
coefficients, FIR taps, detector geometry, SNR snippets — and holds none of
the method's arithmetic (no recursion, no decimation, no projection, no peak
finding).  Recipe: DESIGN.md §"Input recipe"; shapes from SURVEY.md §8(d).
"""
from .configs import CONFIGS, BASE_SEED, config, streams  # noqa: F401
from .gen import (  # noqa: F401
    halfband_taps, detector_geometry, random_bank, chirp_waveform,
    chirp_matched_template, gaussian_strain, inject_chirp, snr_snippets,
    antenna_response, arrival_time, bank_for_config, strain_for_config,
    C_LIGHT, frontend_taps, frontend_psd, frontend_strain, early_warning_bank,
)
