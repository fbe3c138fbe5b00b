"""B200-native hot path of the X-ray pulse-profile forward model of arxiv/paper_2510_07764.

Thin Python binding of the C ABI in include/ppm.h (argument marshalling only; every step of the
path runs in the CUDA kernels of csrc/).  PyTorch supplies device memory and streams.  There is no
CPU fallback: importing works anywhere the library can be built or found, every compute call
raises PPMError when no CUDA device / library is usable.
"""
from .binding import (PPM, PPMError, EXPORTS, lib_path, load_library, measure_fp64_peak,  # noqa: F401
                      loglike_noalloc, NOALLOC_MAX_BATCH,
                      EMISSION_BLACKBODY, EMISSION_TABLE_CUBIC, EMISSION_TABLE_MIXED, EMISSION_TABLE_CUBIC_LINEDGE,
                      EMISSION_TABLE_CUBIC_CLIP)
