"""B200-native hot path of the gateau observation simulator (arXiv 2604.23305).

`workloads` makes the seeded synthetic inputs; `binding` is the thin ctypes layer over
the C ABI in include/gateau_b200.h (libgateau_b200.so, hand-written sm_100a kernels).
Nothing is loaded at import time; the CUDA library is opened on first use and the
binding fails loudly if it is missing.
"""
__all__ = ["workloads", "binding"]
