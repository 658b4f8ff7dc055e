"""B200-native SNAP bispectrum grid descriptors (the MALA inference hot path, arXiv 2411.19617).

`snap` is the ctypes binding of the C-ABI CUDA library (include/mala_snap.h); `workloads` holds the seeded
synthetic inputs.  Nothing here imports the CPU oracle.
"""
from .snap import (MalaSnap, MalaSnapError, load_library, library_path, mala_last_error,  # noqa: F401
                   mala_snap_clebsch_gordan, mala_snap_fp64_peak, bispectrum_for_workload, MalaMlp,
                   bispectrum_ldos_grid)
