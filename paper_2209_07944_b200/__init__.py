"""paper_2209_07944_b200 — B200-native hot path of JefiPIC (arXiv 2209.07944): the full-space Jefimenko field solve
with its history ring, CIC deposit and Boris push, behind the C-ABI of include/jefi.h.

``jefi`` is the ctypes binding (loads the in-tree ``libjefi.so``; no CPU fallback), ``workloads`` the seeded
synthetic inputs, ``build`` the nvcc build step.  Importing the package does not load the CUDA library.
"""
from . import workloads  # noqa: F401

__all__ = ["jefi", "workloads", "build"]
