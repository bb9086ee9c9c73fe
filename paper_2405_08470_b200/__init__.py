"""B200-native all-mode sparse MTTKRP with dynamic tensor remapping (arxiv 2405.08470).

The product is the C-ABI shared library `libmttkrp_b200.so` (include/mttkrp.h, sources under
csrc/); this package is its thin ctypes binding.  Names mirror the C entry points.
"""
from .binding import (EXPORTS, LIB_PATH, Info, Mttkrp, MttkrpError, load_library, mttkrp_workspace_bytes, version)
from .cpd import cpd_als

__all__ = ["cpd_als", "EXPORTS", "LIB_PATH", "Info", "Mttkrp", "MttkrpError", "load_library", "mttkrp_workspace_bytes", "version"]
