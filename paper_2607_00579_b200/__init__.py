"""B200-native (sm_100a) hot path of EPO -- Edge-based Pose Optimization (arxiv 2607.00579).

The product is the CUDA library `libepo.so` behind the C ABI in include/epo.h; this package is only
its build script and a ctypes binding with the same names.  There is no CPU fallback.
"""
from .binding import (Epo, edt_no_alloc, EDT_NO_ALLOC_MAX_PIXELS, EpoConfig, EpoError, epo_config_default, lib, load_library, LIB_PATH, SYMBOLS,  # noqa: F401
                      EPO_OK, EPO_ERR_INVALID_ARG, EPO_ERR_BAD_STATE, EPO_ERR_OUT_OF_MEMORY, EPO_ERR_CUDA,
                      EPO_ERR_UNSUPPORTED)
