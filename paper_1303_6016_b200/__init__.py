"""gfmc-b200: B200-native (sm_100a, fp64) hot path of the O(N) Green-function-based Monte Carlo method for the
3D double-exchange model (arXiv:1303.6016).  The product is libgfmc.so (include/gfmc.h); this package holds
its CUDA sources (csrc/), the ctypes binding with the same names (binding.py), the in-tree build step
(build.py) and the seeded workload generator (workload.py)."""
from . import workload  # noqa: F401
from .binding import *  # noqa: F401,F403
from .binding import EXPORTS, LIB_PATH, Context, GfmcError, load_library  # noqa: F401
