"""paper_1705_02876_b200 -- B200-native batched Kalman-filter track fitting (arXiv:1705.02876).

The product is the C-ABI shared library `libkf_b200.so` (include/kf_b200.h) built from `csrc/`;
this package is the thin ctypes binding with the same call names.  There is no CPU fallback:
without the built library, or without a CUDA device, the calls raise.
"""
from .binding import (KFContext, KFError, Bins, Geometry, Graph, abi_version, lib_path, load_library,
                      strerror, OPT_PAIR_MIN_TRACKS, OPT_REFIT_PAIR_MASKED, OPT_BIN_FORM, BIN_FORM_AUTO,
                      BIN_FORM_FIVE_LAUNCH, BIN_FORM_CHUNKED, STATIC_MAX_CANDIDATES, ERR_TOO_LARGE, STATUS_BAD_CHARGE, STATUS_NONFINITE, STATUS_OUTSIDE, STATUS_PROP_FAIL, STATUS_S_NOT_PD)

__all__ = ["KFContext", "KFError", "Bins", "Geometry", "Graph", "abi_version", "lib_path", "load_library",
           "strerror", "OPT_PAIR_MIN_TRACKS", "OPT_REFIT_PAIR_MASKED", "OPT_BIN_FORM", "BIN_FORM_AUTO",
           "BIN_FORM_FIVE_LAUNCH", "BIN_FORM_CHUNKED", "STATIC_MAX_CANDIDATES", "ERR_TOO_LARGE", "STATUS_BAD_CHARGE", "STATUS_NONFINITE", "STATUS_OUTSIDE", "STATUS_PROP_FAIL", "STATUS_S_NOT_PD"]
