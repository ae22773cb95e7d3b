"""paper_1405_4524_b200 -- B200-native (sm_100a) Wilson-clover Dslash + batched mixed-precision
BiCGStab + Z4 noise fill: the data-parallel hot path of arXiv:1405.4524.

``from paper_1405_4524_b200 import binding`` gives the thin ctypes layer over the C-ABI library
declared in ``include/clover.h``; importing it fails loudly if the CUDA library is not built.
``workloads`` holds the seeded synthetic inputs only (no arithmetic of the method).
"""
