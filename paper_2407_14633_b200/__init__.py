"""B200-native NEGF charge / transmission / Broyden hot path (arXiv 2407.14633).

The product is ``libnegf_b200.so`` (hand-written sm_100a CUDA behind the C-ABI of
``include/negf.h``); this package holds its sources (``csrc/``), the in-tree
build step (``build.py``) and a ctypes binding with the same call names
(``binding.py``).  Nothing here falls back to the CPU.
"""
from .binding import (  # noqa: F401
    Broyden,
    Negf,
    NegfError,
    EXPORTED_SYMBOLS,
    load_library,
    broyden_residual_noalloc,
    NEGF_NOALLOC_MAX_LEN,
    negf_fp64_peak,
    negf_version,
)
