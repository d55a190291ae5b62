"""B200-native (sm_100a) 3-centre Coulomb integrals (X|ab) and integral-direct DF-J — arxiv 2210.03192 hot path.

``paper_2210_03192_b200.lx`` is the thin Python binding of the C-ABI library ``liblx.so`` (include/lx.h): argument
marshalling only; every step of the path runs in the CUDA kernels under ``csrc/``.  Importing the binding fails
loudly when the library has not been built (``python -m paper_2210_03192_b200.build``); there is no CPU fallback.
"""
__all__ = ["lx", "build"]
