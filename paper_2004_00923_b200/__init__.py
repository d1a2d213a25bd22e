"""paper_2004_00923_b200 -- B200-native (sm_100a) hot path of arXiv 2004.00923.

Thin Python binding over the C ABI in include/holo.h (argument marshalling only; every step of the
path runs in the CUDA kernels under csrc/).  PyTorch is used for device memory and streams.
There is NO CPU fallback: importing `binding` without the built library, or creating a handle
without a CUDA device, raises.
"""
from .binding import (Holo, normalize_static, load_library, library_path, HoloError,  # noqa: F401
                      HOLO_OK, HOLO_ERR_ARG, HOLO_ERR_ALLOC, HOLO_ERR_CUDA, HOLO_ERR_STATE, HOLO_ERR_NOCONV,
                      HOLO_WS_SUM, HOLO_WS_H, HOLO_WS_C, HOLO_WS_EVALS, HOLO_WS_V, HOLO_WS_STATUS,
                      HOLO_WS_QX, HOLO_WS_QY, EXPORTED_SYMBOLS)
