"""B200-native Soft-DTW value / gradient / barycenter hot path (arXiv 2404.12134, section 3.3).

Layout: ``csrc/`` holds the hand-written sm_100a CUDA kernels and the C-ABI
(``include/sdtw.h``); ``binding`` is the thin ctypes binding with the same names;
``synth`` draws the seeded synthetic inputs; ``dist`` shards pairs over ranks.
Importing the package does not load the CUDA library; ``binding`` does, and fails loudly
if ``libsdtw.so`` has not been built (``python -m paper_2404_12134_b200.build``).
"""
__version__ = "0.1.0"
