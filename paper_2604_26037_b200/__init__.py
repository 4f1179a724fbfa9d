"""paper_2604_26037_b200 -- B200-native R-ChFSI filter hot path of PAW-FE (arxiv/paper_2604_26037).

The product is ``libpawfe.so`` (C ABI in ``include/pawfe.h``, CUDA sources in ``csrc/``) plus this thin
binding.  There is no CPU fallback: constructing a ``Context`` without the built library or without an
sm_100 GPU raises ``PawfeError``.
"""
from .binding import (  # noqa: F401
    Context, PawfeError, load_library, context_from_system, SYMBOLS, LIB_PATH,
    FP64, FP32, TF32, PREC, PERIODIC, DIRICHLET,
)
