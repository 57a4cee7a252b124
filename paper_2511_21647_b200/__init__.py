"""B200-native (sm_100a) RCA projection beamformer -- the Stage-1 hot path of arxiv 2511.21647.

The product is the C-ABI library declared in include/ulm_rca.h (built by ``paper_2511_21647_b200.build``
into ``libulm_rca.so``); this package is its thin ctypes binding.
"""
from .binding import EXPORTS, Plan, UlmRcaError, fp32_peak_tflops, fold_probe, library_path, load, localize_static, ring_probe  # noqa: F401
