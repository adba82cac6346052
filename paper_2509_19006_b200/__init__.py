"""B200-native BatchTNMC hot path (arXiv 2509.19006): C-ABI library `libtnmc.so` + ctypes binding.

`from paper_2509_19006_b200 import tnmc` loads (building if needed) the CUDA library; see
include/tnmc.h for the boundary and DESIGN.md for the design.  There is no CPU fallback.
"""
__all__ = ["build", "tnmc"]
