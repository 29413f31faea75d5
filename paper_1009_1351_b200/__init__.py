"""paper_1009_1351_b200 -- B200-native (sm_100a) hot path of "Low-dose 4DCT Reconstruction via
Temporal Nonlocal Means" (arxiv 1009.1351).

The product is the C-ABI CUDA library `libtnlm.so` (include/tnlm.h).  This package is a thin
ctypes binding with the same names: it marshals arguments only -- torch tensors supply device
memory and streams, every step of the path runs in the library's kernels.  There is no CPU
fallback: if the library is missing or no CUDA device is present the calls fail loudly.
"""
from .binding import (Geometry, Handle, TnlmError, cgls_step, create, lib_path, library,  # noqa: F401
                      backproject, project, reconstruct, regularize_step, reconstruct_host,
                      regularize_step_host, version, profile_kernels, kernel_times, fbp_init, fma_peak,
                      reserve, set_option, regularize_step_noalloc, NOALLOC_MAX_PIXELS)
