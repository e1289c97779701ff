"""B200-native quench-simulation hot path (after arXiv:2403.07666): CUDA library + thin binding.

``QS`` is the handle class (see binding.py); ``build()`` compiles libqs.so in-tree for sm_100a.
Nothing here imports the CPU oracle; without a CUDA device ``QS(...)`` raises.
"""
from .build import build  # noqa: F401
from .binding import QS, QsError, load_library, SYMBOLS, fp64_peak, pair_eval, issue_probe  # noqa: F401
from .binding import matvec_noalloc, NOALLOC_MAX_RINGS  # noqa: F401
