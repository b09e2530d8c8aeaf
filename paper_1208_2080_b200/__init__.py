"""sw-b200: Swendsen-Wang multi-cluster sweeps of the 2D q-state Potts model on one NVIDIA B200.

The product is the C-ABI library `libsw.so` (include/sw.h, csrc/) and the thin ctypes
binding in `binding.py`.  Importing this package does not load the library; creating a
`SwendsenWang` object does, and fails loudly if it has not been built or no GPU is present.
"""
__all__ = ["binding", "build", "workloads"]
