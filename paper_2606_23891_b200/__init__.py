"""B200-native hot path of the SPH GPU-offload pipeline of arxiv/paper_2606_23891.

The product is libsph_b200.so (hand-written CUDA for sm_100a behind the C ABI in
include/sph_b200.h).  This package is the thin Python binding: same names, argument
marshalling only; PyTorch supplies device / pinned memory and streams.
"""
from .binding import *  # noqa: F401,F403
from .binding import __all__  # noqa: F401
