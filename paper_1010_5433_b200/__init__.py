"""B200-native staggered Dslash + multi-shift CG (arxiv 1010.5433 hot path).

Thin Python binding over the C ABI in include/stag.h (libstag_b200.so, hand-written sm_100a
CUDA).  Argument marshalling only: every step of the path runs in the library's kernels.
PyTorch is used for device memory and streams.  There is no CPU fallback: importing the
binding without a built library raises.
"""
from .binding import (  # noqa: F401
    F64, F32, F64_SPLIT, RECON18, RECON12, MAX_SHIFTS, MAX_RHS, OK, ERR_BADARG, ERR_UNSUPPORTED, ERR_CUDA,
    ERR_NOT_SU3, ERR_NOTCONV, ERR_BREAKDOWN, ERR_SCRATCH_LIMIT, FORCE_STATIC_BYTES, StagError, CgInfo, PolishInfo, MixedInfo, Stag, lib, strerror, SYMBOLS,
)
