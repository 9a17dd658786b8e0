"""B200-native Lagrangian-Eulerian coupling step of the matrix-free immersed boundary method
(arXiv 2503.22695): FE nodal force -> spread -> interpolate, fp64, sm_100a CUDA behind a C ABI.

`workloads` (input generators) imports without the CUDA library; everything in `ibcouple`
loads `libibcouple.so` and fails loudly if it is missing.
"""
__all__ = ["workloads", "ibcouple", "build"]
