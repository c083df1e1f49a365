"""B200-native checkerboard Metropolis for the 2D Ising and Blume-Capel models.

The product is the C-ABI CUDA library `liblattice.so` (include/lattice.h, csrc/); this package
is its thin Python binding plus the seeded workload definitions.  There is no CPU fallback.
"""
from .binding import (BLUME_CAPEL, ISING, Lattice, LatticeBatch, LatticeError, energy, lib, state_bytes,
                      thresholds, thresholds64, xi)
from .buildlib import build
from . import replicas, workloads

__all__ = ["ISING", "BLUME_CAPEL", "Lattice", "LatticeBatch", "LatticeError", "energy", "lib", "state_bytes",
           "thresholds", "thresholds64", "xi", "build", "workloads", "replicas"]
