"""B200-native online TRD tracking step of arXiv 2003.03174 (§3).

The product is the C-ABI library built from ``csrc/`` (declared in ``include/trdmatch.h``);
``binding`` is the thin ctypes layer with the same names.  ``workloads`` holds the seeded
synthetic inputs shared by the oracle's tests and the CUDA path's tests and bench.
"""
__all__ = ["binding", "build", "workloads"]
