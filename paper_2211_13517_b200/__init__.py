"""B200-native Fourier Domain Acceleration Search hot path (arxiv 2211.13517).

Importing this package does not load the CUDA library; ``paper_2211_13517_b200.fdas`` does,
and fails loudly if ``libfdas.so`` has not been built (``python __graft_entry__.py``).
"""
__all__ = ["inputs"]
