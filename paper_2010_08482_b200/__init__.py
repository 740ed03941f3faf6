"""B200-native CT-HYB local-trace library (arXiv:2010.08482, Eq. 65): Python face of libctqmc_b200.so.

Everything here is argument marshalling around the C ABI of include/ctqmc.h; the names are the C names.
"""
from . import binding  # noqa: F401
from .binding import CtqmcError, EXPORTS, ImpurityHandle, LIB_PATH, library  # noqa: F401

# every C name of include/ctqmc.h that the binding mirrors (constants CTQMC_*, functions ctqmc_*)
for _n in dir(binding):
    if _n.startswith(("CTQMC_", "ctqmc_")):
        globals()[_n] = getattr(binding, _n)
del _n
