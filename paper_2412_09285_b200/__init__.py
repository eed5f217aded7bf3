"""B200-native Free-Energy Machine (arxiv 2412.09285) annealing path.

``workloads`` (seeded numpy input generators) imports without the CUDA library;
``fem`` (the binding of include/fem.h) loads ``csrc/libfem_b200.so`` and fails loudly
if it is missing -- there is no CPU fallback.
"""
__all__ = ["workloads", "fem"]
