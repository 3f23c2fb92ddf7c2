"""B200-native multimode CHFPE hot path (arXiv 2509.25840): thin Python binding over libchfpe.so.

Argument marshalling only -- every step of the path runs in the hand-written sm_100a kernels behind the
C-ABI of ``include/chfpe.h``.  PyTorch is used for device memory (the workspace tensor) and streams.
There is no CPU fallback: constructing a ``CHFPE`` without the CUDA library or without a GPU raises.
"""
from .binding import (CHFPE, Hermite, hermite_workspace_bytes, ChfpeError, lib, make_observable, workspace_bytes, spectrum_1d, spectrum_2d,  # noqa: F401
                      spectrum_2d_static_device, SPECTRUM_STATIC_MAX,
                      EXPORTED_SYMBOLS)
