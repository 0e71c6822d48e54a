"""B200-native (sm_100a) dense optical-flow solve of arxiv/paper_1306_2461 (Gautier & Aider).

The product is the C-ABI shared library built from ``csrc/`` (declared in ``include/optflow.h``);
``binding`` is a thin ctypes layer with the same names.  ``synthetic`` makes seeded inputs only.
There is no CPU fallback: every call raises if the CUDA library is missing.
"""
__all__ = ["binding", "synthetic", "build"]
