"""B200-native per-timestep uniform-grid cell update of the QUOKKA method (arXiv:2110.01792).

The product is the C-ABI library built from csrc/ (include/qk.h); `binding` is its thin
ctypes wrapper and `inputs` the seeded synthetic workloads.  Nothing here imports oracle/.
"""
__all__ = ["binding", "inputs", "build"]
