"""paper_2012_00963_b200 -- B200-native Monte-Carlo PDV spectrum (arXiv 2012.00963, section II.B).

Thin Python binding over the C-ABI shared library `libpdv_b200.so` (include/pdv.h).  The names mirror the C
entry points; all computation happens in hand-written CUDA kernels for sm_100a.  No CPU fallback.
"""
from ._binding import (  # noqa: F401
    EXPORTS, LIB_PATH, PDV_MAX_BINS, PDV_MAX_CLASSES, PDV_STATIC_SCRATCH_BYTES, PEAK_DTYPE, STATS_DTYPE, TRACE_DTYPE, Cloud, PdvError, RunResult, lib,
    pdv_cloud_create, pdv_issue_peaks, pdv_last_launch_info, pdv_lognormal_classes, pdv_mc_run, pdv_mc_run_device, pdv_mc_run_static,
    pdv_mc_trace, pdv_phase_sampling_check, pdv_philox_blocks, pdv_spectrogram, pdv_spectrum_peaks, pdv_version,
)
