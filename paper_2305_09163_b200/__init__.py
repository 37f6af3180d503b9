"""B200-native hot path of arxiv 2305.09163 (MFC): RHS of the 5-equation model behind a C ABI.

    binding    thin ctypes layer over libmfc_b200.so (include/mfc.h); no CPU fallback
    build      nvcc build of the library for sm_100a
    workloads  seeded synthetic inputs shaped like the paper's workloads (shared with the tests' oracle)
"""
__all__ = ["binding", "build", "workloads"]
