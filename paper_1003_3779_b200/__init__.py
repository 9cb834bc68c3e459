"""paper_1003_3779_b200 — B200-native coined quantum-walk stepper (arXiv 1003.3779 hot path).

The product is the C-ABI library ``libqw.so`` built from ``csrc/`` (declared in
``include/qw.h``); ``binding`` is a thin ctypes front end with the same names and
``inputs`` holds the seeded synthetic workloads.  Nothing here falls back to a CPU
implementation: calling into the library without the built CUDA extension raises.
"""
__all__ = ["binding", "inputs", "build"]
