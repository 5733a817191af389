"""B200-native hot path of Splaxel's pixel-level scheme (arxiv/paper_2606_18588).

``binding`` is the thin ctypes layer over ``libsplx.so`` (the C-ABI of
``include/splx.h``); ``scenes`` holds the seeded synthetic input generators
(no method arithmetic).  Importing this package does not load the CUDA
library; the first ``binding`` call does, and fails loudly if it is missing.
"""
__all__ = ["binding", "scenes"]
