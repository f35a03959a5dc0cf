"""B200-native Swendsen-Wang multi-cluster sweep (arXiv 1202.0635) behind the C ABI of include/sw.h.

``binding`` is the ctypes layer over ``libsw.so`` (hand-written CUDA for sm_100a, no CPU fallback);
``workloads`` holds the seeded synthetic workloads; ``build`` compiles the library in-tree.
"""
from . import workloads  # noqa: F401  (no native code needed)

__all__ = ["binding", "build", "workloads"]
