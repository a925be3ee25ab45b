"""nkb200 — batched RBM local energies for lattice spin Hamiltonians on one B200 (sm_100a).

Thin Python binding over the C-ABI library `libnkb200.so` (include/nkb200.h).  Importing the package is
cheap and needs no GPU; `load()` (or the first call) opens the shared library and fails loudly if absent.
"""
from .binding import *            # noqa: F401,F403
from .binding import __all__      # noqa: F401
