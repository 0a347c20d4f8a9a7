"""paper_1309_2256_b200 -- B200-native twisted-mass dslash / MdagM / CG / loop library (arxiv/paper_1309_2256 hot path).

Thin ctypes binding of libtm_b200.so (C ABI in include/tm.h).  Argument marshalling only: every step of the path
runs in the CUDA kernels under csrc/.  PyTorch is used for device memory and streams, nothing else.
There is no CPU fallback: importing works without a GPU (so the ABI can be checked), compute calls need one.
"""
from .binding import *  # noqa: F401,F403
from .binding import __all__  # noqa: F401
