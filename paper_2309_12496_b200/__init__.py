"""paper_2309_12496_b200 -- B200-native per-photon optical propagation (arXiv:2309.12496).

csrc/   CUDA kernels + the C ABI of include/opx.h (and the debug exports of include/opx_debug.h)  (-> lib/libopx.so, built by build.py)
opx.py  thin ctypes/torch binding with the same names

Nothing here imports the oracle, and there is no CPU fallback.
"""
from .opx import (DEBUG_EXPORTS, EXPORTS, FLAG_NO_EFFICIENCY, LIB_PATH, STATE_NAMES, TABLE_HISTOGRAM, TABLE_LINEAR, OpxError, Scene, alloc_host_detected, alloc_host_records,  # noqa: F401
                  emit_cherenkov, last_kernel, launch_count, load_library, measure_fp32_peak, upload_track_steps)
