"""paper_1801_06364_b200 — B200-native (sm_100a) time stepper for the pseudospectral P_N radiative transport method
of Powell, Cox & Arridge (arXiv:1801.06364).  The product is the C-ABI library of include/rte.h (built from csrc/);
this package is the thin binding over it.  Importing it fails loudly when the CUDA library has not been built."""
from .binding import *  # noqa: F401,F403
from .binding import EXPORTED, LIB_PATH, Context, RteError, rte_grid, rte_media, rte_pml  # noqa: F401
