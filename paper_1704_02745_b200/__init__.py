"""B200-native Jacobi-PCG for the linear finite-difference Poisson-Boltzmann equation.

Thin Python binding over the C ABI of include/pb.h (libpb.so, hand-written sm_100a kernels).
Argument marshalling only: every step of the method runs in the CUDA library.  There is no
CPU fallback -- importing works without a GPU, but every compute call raises if the library
or a CUDA device is missing.
"""
from .binding import (  # noqa: F401
    PB_DEVICE,
    PB_F32,
    PB_F64,
    PB_HOST,
    OPTIONS,
    PBError,
    PBSolver,
    STATUS_NAMES,
    lib_path,
    load_library,
    pb_strerror,
    residual_noalloc,
    NOALLOC_MAX_ROWS,
)
