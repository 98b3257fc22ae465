"""B200-native sparse lattice-Boltzmann site update (arxiv 1906.11925, HemeLB-style).

The product is the C-ABI library ``libhlb.so`` (include/hlb.h, csrc/); this package is its
in-tree build plus a thin ctypes binding with the same names. Importing the package builds
and loads the library and fails loudly if that is impossible -- there is no CPU fallback.
"""
from .binding import *  # noqa: F401,F403
from .binding import Geometry, HlbError, LIB_PATH, EXPORTED, hlb_params, hlb_view, make_view  # noqa: F401
from .metrics import msups, sups, BYTES_PER_SITE, algorithmic_bytes_per_site, moved_bytes_per_site  # noqa: F401
