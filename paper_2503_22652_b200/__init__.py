"""B200-native R-ChFSI filter library (arxiv 2503.22652): Python binding of librchfsi.so.

The product is the CUDA library in csrc/ behind the C ABI of include/rchfsi.h; this package
only marshals arguments.  Importing it does not need a GPU; using it does, and fails loudly
when the library is not built or no device is present (no CPU fallback).
"""
from .binding import (Rchfsi, RchfsiError, RchfsiOperator, RchfsiOptions, RchfsiBounds, load_library, LIB_PATH, SYMBOLS,
                      OK, EINVAL, ENOMEM, ECUDA, ENOTCONVERGED, EBREAKDOWN, FP64, FP32, TF32, BF16,
                      METHOD_CHFSI, METHOD_RCHFSI, OP_DENSE, OP_CSR, OP_FE, USE_FILTER, USE_RAYLEIGH_RITZ,
                      USE_SOLVE, USE_FILTER_HOST, USE_BOUNDS, USE_FILTER_NULL_G, STATIC_MAX_N, static_setup,
                      residual_static)
from .problems import upload_problem

__all__ = ["Rchfsi", "RchfsiError", "RchfsiOperator", "RchfsiOptions", "RchfsiBounds", "load_library", "LIB_PATH", "SYMBOLS",
           "upload_problem", "OK", "EINVAL", "ENOMEM", "ECUDA", "ENOTCONVERGED", "EBREAKDOWN", "FP64", "FP32",
           "TF32", "BF16", "METHOD_CHFSI", "METHOD_RCHFSI", "OP_DENSE", "OP_CSR", "OP_FE", "USE_FILTER",
           "USE_RAYLEIGH_RITZ", "USE_SOLVE", "USE_FILTER_HOST", "USE_BOUNDS", "USE_FILTER_NULL_G", "STATIC_MAX_N",
           "static_setup", "residual_static"]
