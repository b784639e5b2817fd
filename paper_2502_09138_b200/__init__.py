"""paper_2502_09138_b200 -- B200-native TPC sector track finding (arXiv:2502.09138, Table 1: TPC processing).

Thin Python binding over the C ABI in include/tpc_track.h (libtpctrack.so, hand-written CUDA for sm_100a).
Argument marshalling only: every step of the path runs in the library's kernels.  There is no CPU fallback:
importing the binding without the built library, or calling it without a CUDA device, raises.
"""
from .binding import (Geometry, Params, Tracker, TrackRec, TracksOut, TRACK_DTYPE, lib_path, load_library,  # noqa: F401
                      declared_symbols, rans_alloc, rans_encode_static, RANS_STATIC_SCRATCH_BYTES)
