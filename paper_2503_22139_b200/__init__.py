"""gsvox: B200-native (sm_100a) differentiable 3D Gaussian voxelizer — the data-parallel hot
path of PMF-STGR (arXiv 2503.22139, Eq. 4-5).  See DESIGN.md and include/gsvox.h."""
from .binding import (EXPORTS, PROBE_EXPORTS, K_NAMES, LIB_PATH, GsvoxError, GsvoxGrid, GsvoxStatus, Plan, Splatter, lib,
                      make_grid, mbc_combine_backward, mbc_combine_forward, probe_lib, probe_peaks, project_backward, project_forward, project_forward_static, warp_backward,
                      warp_forward)

__all__ = ["EXPORTS", "PROBE_EXPORTS", "K_NAMES", "LIB_PATH", "GsvoxError", "GsvoxGrid", "GsvoxStatus", "Plan", "Splatter", "lib",
           "make_grid", "mbc_combine_backward", "mbc_combine_forward", "probe_lib", "probe_peaks", "project_backward", "project_forward", "project_forward_static", "warp_backward", "warp_forward"]
from .pipeline import Stage3Step  # noqa: E402

__all__.append("Stage3Step")
