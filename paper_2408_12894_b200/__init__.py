"""B200-native forward rasterizer for multi-level 3D Gaussian sets (FLoD, arXiv 2408.12894).

The product is `libflod.so` (hand-written sm_100a CUDA behind the C ABI of include/flod.h); this package is
the thin ctypes binding over it.  There is no CPU fallback: without the built library every entry point raises.
Build with `python -m paper_2408_12894_b200.build` (or `__graft_entry__.build()`).
"""
from .binding import (overlap_prune, overlap_prune_static, overlap_prune_static_max_n, PAIR_RULE_BOX, PAIR_RULE_ELLIPSE, FLOD_OPT_COUNT, FLOD_OPT_DEBUG, FLOD_OPT_PROFILE, FLOD_OPT_SMALL_WINDOWS, FLOD_OPT_FULL_SORT, FlodError, Renderer, abi_symbols,
                      load_library)

__all__ = ["overlap_prune", "overlap_prune_static", "overlap_prune_static_max_n", "PAIR_RULE_BOX", "PAIR_RULE_ELLIPSE", "Renderer", "FlodError", "load_library", "abi_symbols",
           "FLOD_OPT_DEBUG", "FLOD_OPT_PROFILE", "FLOD_OPT_COUNT", "FLOD_OPT_SMALL_WINDOWS", "FLOD_OPT_FULL_SORT"]
