"""paper_1411_3396_b200 -- B200-native short-range particle-particle force solver (HACC's short-range
hot path as named by arXiv:1411.3396, Sec. 2): chaining-mesh binning, PP force, sub-cycled kick.

Layout: `csrc/` CUDA kernels + the C ABI of include/srpp.h (built in-tree as libsrpp.so),
`binding.py` thin ctypes/torch marshalling, `workloads.py` seeded synthetic inputs, `build.py`.
Importing this package does not load the CUDA library; `binding.load()` / `Solver` do, and raise
if it is missing (there is no CPU fallback).
"""
__all__ = ["binding", "workloads", "build"]
