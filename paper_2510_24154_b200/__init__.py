"""B200-native hot path of ARCHER-EPID (arxiv 2510.24154): coupled photon/electron Monte Carlo
transport through a voxel phantom and a multi-layer EPID, hand-written CUDA for sm_100a behind
the C-ABI of include/aepid.h.  See DESIGN.md.  There is no CPU fallback."""
from .binding import (AepidError, Dims, Engine, LIB_PATH, LEDGER_NAMES, COUNTER_NAMES, EXPORTS,  # noqa: F401
                      load_library, workspace_bytes, gamma_of_upsampled_static)

__all__ = ["AepidError", "Dims", "Engine", "LIB_PATH", "LEDGER_NAMES", "COUNTER_NAMES", "EXPORTS",
           "load_library", "workspace_bytes", "gamma_of_upsampled_static"]
