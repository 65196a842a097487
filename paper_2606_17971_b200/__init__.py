"""B200-native hot path of arxiv/paper_2606_17971 (reference-space deflated CG inside PDAS).

The product is the CUDA library `librefdef_b200.so` (C ABI: include/refdef.h, sources: csrc/);
this package is its thin Python binding (argument marshalling only).  There is no CPU fallback:
importing works anywhere, creating a context without the library or without a CUDA device raises.
"""
from .binding import (  # noqa: F401
    RefDef, RefDefError, Options, JACOBI_CG, REFDEF, ZEROEXT, INIT_PAPER, INIT_ALL_ACTIVE,
    INIT_ALL_INACTIVE, INIT_GIVEN, STATUS_NAMES, load_library, exported_symbols, LIB_PATH, NOALLOC_MAX_N,
)
