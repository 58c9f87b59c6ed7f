"""B200-native red-black checkerboard Metropolis for classical Heisenberg spins (arXiv 2103.03517).

The product is the C-ABI shared library ``libmc_b200.so`` (hand-written CUDA for sm_100a, declared in
``include/mc.h``); :mod:`paper_2103_03517_b200.binding` is a thin ctypes layer over it with the same
names.  Importing this package does not load the CUDA library; the first use of the binding does, and
fails loudly if it is missing -- there is no CPU fallback.
"""

__all__ = ["binding", "inputs", "build", "harness"]
