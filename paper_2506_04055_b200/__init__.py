"""B200-native PaiNN energy / force / virial hot path (arXiv 2506.04055 deployment path, rebuilt for sm_100a).

Thin Python binding over the C ABI of ``include/mlp.h``: argument marshalling only -- every step of the path
runs in the CUDA kernels of ``csrc/``.  PyTorch is used for device memory and streams.  There is no CPU
fallback: if the shared library is missing or no CUDA device is present, calls raise.
"""
from .binding import (  # noqa: F401
    MLPError, Model, lib_path, load_library, version, debug_gemm, measure_row_gather, row_offsets, row_offsets_into,
    ROW_OFFSETS_STATIC_MAX, EXPORTED_SYMBOLS,
)
