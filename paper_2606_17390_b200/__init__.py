"""B200-native fem_assemble (arxiv 2606.17390 hot path).  Thin ctypes binding over libfem_b200.so.

Every step of the path runs in the CUDA kernels of csrc/; this module only marshals arguments
(torch tensors -> device pointers, the current torch stream -> cuda_stream).  There is no CPU fallback:
if the shared library is missing, or no CUDA device is visible, calls raise.
"""
from .binding import (FemContext, FemError, FemOptions, FemStats, FemNewtonOptions, FemNewtonReport, NPAR, hill_from_lankford, lib, lib_path,  # noqa: F401
                      mat_from_desc, mat_record, barlat_record, NBARLAT, probe_fp64_peak, ABI_SYMBOLS)
