"""B200-native LLOID matched-filter hot path (arXiv:2410.16416) — Python side.

``workloads``  seeded synthetic banks and strain (numpy only; also used by the oracle's tests)
``binding``    ctypes binding of the C ABI in include/lloid.h (needs the built liblloid.so)
``build``      nvcc build of csrc/ into liblloid.so for sm_100a
Importing the package itself loads nothing heavy.
"""
__all__ = ["workloads", "binding", "build"]
