"""paper_2604_15380_b200 — B200-native batched PaiNN energy+force evaluation (the hot path of
arxiv/paper_2604_15380's multi-task atomistic graph foundation model).

The product is the C-ABI library `libpnn.so` (hand-written sm_100a CUDA; declarations in include/pnn.h).
This package is its thin Python binding: same entry-point names, argument marshalling only.  It fails
loudly if the library has not been built (python -m paper_2604_15380_b200.build); there is no CPU fallback.
"""
from .binding import *  # noqa: F401,F403
from .binding import __all__  # noqa: F401
