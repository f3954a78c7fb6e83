"""paper_1104_3408_b200 -- thin Python binding of libspshell (include/spshell.h).

Argument marshalling only: every step of the hot path (gradient, Yn tensor filter, wave RHS)
runs in the hand-written sm_100a kernels of csrc/.  PyTorch is used for device memory and
streams.  There is no CPU fallback: importing works anywhere (so the ABI can be inspected), but
every compute call raises unless the CUDA library is built and a CUDA device is present.
"""
from .binding import (SpError, Shell, lib, library_path, probe_fp64_peak, status_string,  # noqa: F401
                      EXPORTED_SYMBOLS, launch_count)
