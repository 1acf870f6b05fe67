"""B200-native AVU-GSR hot path (aprod1, aprod2, LSQR) -- thin Python binding of libgsr.so.

Every step of the path runs in the hand-written sm_100a kernels behind the C ABI declared
in include/gsr.h; this package only marshals arguments (torch tensors -> device pointers,
the current torch stream -> cudaStream_t).  There is no CPU fallback: if libgsr.so is not
built, or no CUDA device is present, the calls raise.
"""
from .binding import (GsrError, GsrSystem, LsqrResult, gsr_aprod1, gsr_aprod2, gsr_create,  # noqa: F401
                      gsr_destroy, gsr_lsqr, gsr_lsqr_host, gsr_version, lib, lib_path)
