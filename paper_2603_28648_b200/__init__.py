"""B200-native two-site DMRG hot path (H_eff.psi, Davidson, renormalization) of arxiv/paper_2603_28648.

The product is the C-ABI library `libdmrg_b200.so` (include/dmrg.h, csrc/); this package holds the
thin ctypes binding with the same call names and the build step.
"""
from .binding import *  # noqa: F401,F403
from .binding import Dmrg, DmrgError, load_library, LIB_PATH, EXPORTS, dots_noalloc  # noqa: F401
from .build import build_library  # noqa: F401
