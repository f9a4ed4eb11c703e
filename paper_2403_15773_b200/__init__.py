"""B200-native thread-safe lattice Boltzmann (TSLB) two-component time step (arxiv 2403.15773).

`tslb` is the ctypes binding of the C-ABI CUDA library (include/tslb.h); `inputs` holds the
seeded synthetic workload generators.  Nothing is loaded at import time; the CUDA library is
opened on first use and its absence is a hard error (there is no CPU fallback).
"""
__all__ = ["tslb", "inputs"]
