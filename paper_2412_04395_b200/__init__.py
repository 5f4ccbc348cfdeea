"""B200-native RK3 dynamical-core step after the ERF paper (arXiv 2412.04395).

The product is the C-ABI library ``liberf_b200.so`` (csrc/, include/erf_b200.h)
and the thin ctypes binding in :mod:`paper_2412_04395_b200.binding`.
:mod:`paper_2412_04395_b200.workloads` holds the seeded synthetic inputs.
"""
__all__ = ["binding", "workloads"]
