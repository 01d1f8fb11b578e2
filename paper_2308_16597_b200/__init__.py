"""B200-native hot path of the particle-resolved thermal lattice Boltzmann method of
Xu & Li (arXiv 2308.16597): hand-written sm_100a CUDA kernels behind the C ABI in include/lbm.h.

`binding` is the thin ctypes layer over the C-ABI shared library (argument marshalling only);
`workloads` generates the seeded synthetic inputs.  There is no CPU fallback: importing
`binding.Simulation` without the built library or without a GPU fails loudly.
"""
from . import workloads  # noqa: F401

__all__ = ["workloads"]
