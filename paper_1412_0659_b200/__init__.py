"""B200-native Barnes-Hut tree force (hot path of arxiv 1412.0659, the Bonsai paper).

The product is ``libbhtree.so`` (hand-written CUDA for sm_100a behind the C ABI of
``include/tree.h``).  This package is the thin ctypes binding with the same names; it only
marshals arguments.  There is no CPU fallback: if the CUDA library is missing or no GPU is
present, calls fail loudly.
"""
from .binding import (  # noqa: F401
    Tree,
    TreeError,
    load_library,
    library_path,
    exported_symbols,
    tree_create,
    tree_build,
    tree_force,
    tree_leapfrog,
    tree_destroy,
    tree_energy_static,
    ENERGY_STATIC_MAX_N,
    PHASES,
    FLOP_PP,
    FLOP_PC,
    effective_flops,
)
