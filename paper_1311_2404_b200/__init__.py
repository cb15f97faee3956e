"""B200-native fused lattice Boltzmann stream-and-collide (arXiv 1311.2404 hot path).

The product is the C-ABI CUDA library declared in include/lbm.h (built into
paper_1311_2404_b200/liblbm_b200.so by paper_1311_2404_b200.build) and the thin ctypes binding in
paper_1311_2404_b200.binding.  Importing the package does not load the library; using the
binding without the built library raises (there is no CPU fallback).
"""
__all__ = ["binding", "build", "workloads"]
