"""B200-native hot path of the Fourier-domain jerk search (arXiv 1911.01353).

The compute path lives in ``csrc/`` (CUDA, sm_100a) behind the C-ABI declared in
``include/jerk.h``; ``binding`` is the thin ctypes layer with the same names.
There is no CPU fallback: calls fail loudly if the shared library is missing.
"""
__all__ = ["binding", "build", "shard"]
