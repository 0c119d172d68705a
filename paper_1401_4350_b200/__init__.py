"""paper_1401_4350_b200 -- B200-native VERTEX / EDGE short-range MD force kernels (arXiv 1401.4350).

Thin Python binding over the C ABI of include/md_b200.h (libmd_b200.so, hand-written CUDA for sm_100a).
PyTorch is used for device memory and streams only; there is no CPU or PyTorch fallback: importing
`MDSystem` without the built library raises.
"""
from .binding import (MDSystem, MDError, load_library, STRATEGY, SCATTER, GATHER, ORDER, POT_KIND, library_path,
                      EXPORTED_SYMBOLS, energy_static, ENERGY_STATIC_MAX_N)

__all__ = ["MDSystem", "MDError", "load_library", "STRATEGY", "SCATTER", "GATHER", "ORDER", "POT_KIND", "library_path",
           "EXPORTED_SYMBOLS", "energy_static", "ENERGY_STATIC_MAX_N"]
