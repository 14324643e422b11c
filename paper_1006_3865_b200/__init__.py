"""paper_1006_3865_b200 — B200-native double-checkerboard Metropolis sweep (arXiv 1006.3865).

The product is the C-ABI library `libising_b200.so` (include/ising.h, include/heisenberg.h, csrc/*.cu, sm_100a);
`binding` marshals arguments to it.  Nothing in this package imports `oracle/`.
"""
from .binding import (HEIS_SYMBOLS, Heisenberg, ISING_LAYOUT_BITS, ISING_LAYOUT_I8, ISING_RNG_PLANES, ISING_RNG_WORDS, SYMBOLS, Ising, IsingError,
                      STATIC_MAX_REPLICAS, ising_kernel_launches, ising_overlap_all_static, ising_thresholds, lib, use_torch)

__all__ = ["Heisenberg", "HEIS_SYMBOLS", "Ising", "IsingError", "ISING_LAYOUT_I8", "ISING_LAYOUT_BITS", "ISING_RNG_WORDS", "ISING_RNG_PLANES", "SYMBOLS", "lib",
           "use_torch", "ising_thresholds", "ising_kernel_launches", "ising_overlap_all_static", "STATIC_MAX_REPLICAS"]
