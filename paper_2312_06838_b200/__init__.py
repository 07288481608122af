"""B200-native EdgeConv-GNN inference hot path (arXiv 2312.06838's served model): thin ctypes binding over libgnn.so.

Argument marshalling only -- every step of the path runs in the library's CUDA kernels.  torch is used for device
memory and streams.  There is no CPU fallback: loading fails loudly if libgnn.so is missing.
"""
from .binding import (GnnArch, Model, Batcher, Bdt, GnnError, lib, arch_struct, weights_bytes, strerror, LIB_PATH,  # noqa: F401
                      FP32_VALIDATION, BF16, knn_noalloc)
