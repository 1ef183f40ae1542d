"""alora-b200: the ALM-BM hot path of ALORA (arXiv 2505.15775) as sm_100a CUDA kernels.

``inputs``  -- seeded synthetic problem generators (numpy only, no method arithmetic)
``binding`` -- thin ctypes binding over the C-ABI library ``csrc/libalora.so`` (include/alora.h)
"""
