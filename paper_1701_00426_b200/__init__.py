"""B200-native staggered Dslash / CG / multi-shift CG (arxiv/paper_1701_00426 hot path).

Thin Python binding over the C ABI of include/lqcd.h (liblqcd_b200.so, hand-written CUDA for
sm_100a).  Argument marshalling only: every step of the path runs in the CUDA kernels.  PyTorch
is used by callers for device memory and streams.  There is no CPU fallback: importing works
without a GPU (so that symbols can be checked), but creating a context without one fails loudly.
"""
from .binding import (  # noqa: F401
    LqcdError,
    Lattice,
    lib,
    lib_path,
    F64, F32, RECON_18, RECON_12, EVEN, ODD,
    OK, ERR_ARG, ERR_UNSUPPORTED, ERR_CUDA, ERR_NOT_CONVERGED, ERR_WORKSPACE,
    MAX_SHIFTS,
    version,
    HALO_FN, ALLREDUCE_FN, PHASE_FN,
)
