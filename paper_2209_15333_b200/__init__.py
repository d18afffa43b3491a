"""B200-native RHS / RK3 hot path of the OpenCFD-SCU finite-difference DNS method (arxiv 2209.15333).

`paper_2209_15333_b200.binding` is the thin ctypes layer over the C-ABI CUDA library
(include/ocfd.h, csrc/); `paper_2209_15333_b200.workloads` holds the seeded synthetic input
generators shared by the CUDA path and the test oracle.  Importing this package loads neither.
"""
__all__ = ["binding", "workloads"]
