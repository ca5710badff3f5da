"""B200-native PTEFIT hot path (arxiv 2601.12378): thin Python binding over libptefit.so.

Argument marshalling only -- every step of the Picard iteration runs in the CUDA library
(include/ptefit.h).  There is no CPU fallback: importing works anywhere (so the ABI can be
checked), but creating a handle without a B200 raises.
"""
from .binding import (PtefitError, Reconstructor, load_library, poly_terms,  # noqa: F401
                      ptefit_create, ptefit_destroy, ptefit_reconstruct, ptefit_greens_table, EXPORTED_SYMBOLS, shard_slices)
