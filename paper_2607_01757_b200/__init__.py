"""paper_2607_01757_b200 — B200-native DKD keypoint post-processing + descriptor sampling.

Thin Python binding over the C-ABI of ``include/dkd.h`` (``libdkd.so``, hand-written CUDA for
sm_100a).  Argument marshalling only: every step of the hot path runs in the library's kernels.
PyTorch is used for device memory and streams.  There is no CPU fallback: importing works
anywhere, but creating a context without the library or without a CUDA device raises.
"""
from .binding import (DKD, DKDError, DKDResult, F16, F32, lib_path, load_library,  # noqa: F401
                      EXPORTED_SYMBOLS, MATCH_STATIC_MAX_RECS, match_static)
from .sharding import shard_range, sharded_extract  # noqa: F401

__all__ = ["DKD", "DKDError", "DKDResult", "F16", "F32", "lib_path", "load_library",
           "EXPORTED_SYMBOLS", "MATCH_STATIC_MAX_RECS", "match_static", "shard_range", "sharded_extract"]
