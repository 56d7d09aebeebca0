"""B200-native KBMOD shift-and-stack search hot path (arXiv 2109.03296): Python binding of the C-ABI
library libkbmod_b200.so (include/kbmod_b200.h) plus the seeded synthetic input generators."""
from . import binding  # noqa: F401
from .binding import (ALGO_AUTO, ALGO_DIRECT, ALGO_PRUNED, KbmodError, Plan, SearchParams)  # noqa: F401

# every C entry point under its own name
for _n in binding.EXPORTS:
    if hasattr(binding, _n):
        globals()[_n] = getattr(binding, _n)
del _n
