"""gamer-hydro-b200: the batched relaxing-TVD hydrodynamic update of GAMER (arXiv 0907.3390) for B200 (sm_100a).

The product is the C-ABI library declared in include/gamer_hydro.h (built into this package as
libgamer_hydro.so); `paper_0907_3390_b200.hydro` is the thin Python binding with the same entry points.
Importing the package does not load the library; the first call does, and it fails loudly if the library
is missing (there is no CPU fallback).
"""
__version__ = "0.1.0"
