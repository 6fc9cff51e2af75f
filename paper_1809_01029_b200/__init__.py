"""pyjac-b200: B200-native batched chemical-kinetic source terms and analytical Jacobians
(after pyJac v2, arXiv:1809.01029).  The product is the C-ABI library declared in include/pyjac.h;
this package is its build script and a thin ctypes binding with the same names."""
from .binding import *  # noqa: F401,F403
from .binding import lib, Mechanism, PyjacError, make_desc, LIB_PATH
