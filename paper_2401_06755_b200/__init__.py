"""B200-native multigrid pressure solve and explicit stencil residuals of arxiv/paper_2401_06755.

The product is the C-ABI library libmg_b200.so (include/mg.h, sources under csrc/); this package
is its thin Python binding.  Importing it loads the library and raises if that is impossible.
"""
from .binding import *  # noqa: F401,F403
from .binding import (MgError, MgGrid, MgParams, Solver, EXPORTS, library_path)  # noqa: F401
