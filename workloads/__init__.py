"""Seeded input generators shared by the oracle-side tests and the CUDA-side tests / bench.

Holds none of the method's arithmetic (see generators.py)."""
from .generators import *  # noqa: F401,F403
from .generators import BASE_SEED, DESC_DTYPE, CopyWorkload, ChannelWorkload, GlobalWorkload  # noqa: F401
