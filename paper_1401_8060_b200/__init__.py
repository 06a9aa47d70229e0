"""paper_1401_8060_b200 -- B200-native hot path of all-sky stochtrack (arXiv:1401.8060).

A thin ctypes binding (argument marshalling only) over the C-ABI library
`libstochtrack_b200.so` declared in include/stochtrack.h.  Every step of the path
(template generation, Bezier rasterisation, Eq. 8 scoring, max/argmax/histogram)
runs in hand-written sm_100a CUDA kernels; there is no CPU fallback: importing
`binding` raises if the library has not been built, and every call raises if no
CUDA device is present.
"""
from .binding import (Stochtrack, StError, SearchResult, st_track_params, st_track_words,  # noqa: F401
                      library_path, load_library, exported_symbols,
                      score_random_noalloc, NOALLOC_MAX_PIXELS, NOALLOC_SCRATCH_BYTES,
                      KERNEL_AUTO, KERNEL_TABLE, KERNEL_ROTATION, KERNEL_REINSCH, KERNEL_RANDOM, KERNEL_CHEBYSHEV,
                      NORM_SQRT_N, NORM_MEAN, NORM_INVVAR, FAMILY_QUADRATIC, FAMILY_CUBIC, FAMILY_CHIRP, TAU_GRID, TAU_RANDOM)
