"""B200-native UT decode + Compass tracking (arxiv/paper_2002_11529 hot path).

The product is ``libutcompass.so`` (hand-written CUDA for sm_100a behind the C ABI of
``include/ut_compass.h``).  This package is the thin Python binding: argument marshalling
only -- every step of the path runs in the CUDA kernels.  There is no CPU fallback: importing
``binding`` fails loudly if the library is missing or cannot be loaded.
"""
__version__ = "0.1"
__all__ = ["binding", "build"]
