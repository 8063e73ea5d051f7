"""B200-native (sm_100a) Z-refinement hot path of arXiv 2404.19163.

`binding` is the ctypes layer over libzfac.so (include/zfac.h); `workloads` holds the seeded
synthetic inputs; `build` compiles the library in-tree.  Importing the package does not load
the library; calling into `binding` without it fails loudly (there is no fallback path).
"""
__all__ = ["binding", "workloads", "build"]
