"""B200-native ERI-derivative gradient (arXiv 2407.16586 hot path).

``workload`` (seeded inputs) imports nothing native; ``tdgrad`` is the ctypes binding of the
C-ABI CUDA library and raises if ``libtdgrad.so`` is missing (no CPU fallback).
"""
