"""B200-native hot path of the mixed-variational phononic band-structure method (arXiv:1310.6380).

``libbs.so`` (hand-written sm_100a CUDA behind the C-ABI of ``include/bs.h``) does all the work; this package is the
thin ctypes binding with the same names.  No CPU fallback exists.
"""
from .binding import *  # noqa: F401,F403
from .binding import Cell, BsError, lib, LIB_PATH, SYMBOLS, allocate_workspace  # noqa: F401
