"""B200-native radiation stage of the finite-solid-angle GR transport of White et al.
(arXiv 2302.04283): C-ABI library `librad.so` (csrc/, hand-written CUDA for sm_100a) plus
a thin Python binding (`binding`).  `workloads` holds the seeded synthetic inputs only.

Importing the package does not load the CUDA library; `binding.lib()` does, and raises
if it is missing (there is no CPU fallback).
"""
__all__ = ["binding", "workloads", "build"]
