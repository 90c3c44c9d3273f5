"""B200-native batched rebalancing solver (PRISM hot path): thin Python binding over the C-ABI library."""
from .binding import (Problem, Settings, SolveResult, lib, load_library, version, NRES, RES, STATUS_NAMES)  # noqa: F401
