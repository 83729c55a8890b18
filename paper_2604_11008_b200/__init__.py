"""paper_2604_11008_b200: B200-native particle hot path of LCS.jl (arxiv/paper_2604_11008).

Thin ctypes binding over the C ABI in include/lcs.h (liblcs_b200.so, hand-written CUDA for
sm_100a).  PyTorch is used only for device memory and streams.  There is no CPU fallback: every
entry point fails loudly if the library or a CUDA device is missing.
"""
from .binding import (LCS, LcsError, lib_path, load_library, EXPORTED_SYMBOLS,  # noqa: F401
                      LCS_OK, LCS_ERR_INVALID_ARG, LCS_ERR_STATE, LCS_ERR_CUDA, LCS_ERR_CAPACITY,
                      LCS_ERR_JUMP, LCS_ERR_RANGE, LCS_ERR_NOMEM, LCS_ERR_TOO_LARGE,
                      LCS_PAIR_COUNT_STATIC_MAX_SLOTS)
