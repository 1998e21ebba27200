"""ddamg-b200: the odd-even (Schur-complement) Wilson-clover hot path of DD-alphaAMG
(arXiv:2407.08092) as hand-written CUDA for NVIDIA B200 (sm_100a) behind a C ABI.

``binding.Ddamg`` mirrors include/ddamg.h one to one; ``build.build_library`` compiles
libddamg.so in-tree.  There is no CPU fallback and this package never imports ``oracle``.
"""
from .binding import (  # noqa: F401
    Ddamg, DdamgError, load_library, SYMBOLS, LIB_PATH,
    OK, EINVAL, ENOMEM, ESTATE, ECUDA, ESINGULAR, F32, F64, BC_PERIODIC, BC_ANTIPERIODIC_T,
    SMOOTHER_RICHARDSON, SMOOTHER_GMRES, SMOOTHER_GCR, SMOOTHER_SAP,
)
from .build import build_library  # noqa: F401
