"""paper_2606_00746_b200 -- B200-native GSPN 2D line-scan propagation (libgspn + thin binding).

The product is the C-ABI library `libgspn.so` (include/gspn.h, sources under csrc/); this
package only marshals torch tensors into it.  Build it with `python -m paper_2606_00746_b200.build`.
"""
from .binding import (  # noqa: F401
    BF16, DIR_ALL, DIR_BT, DIR_LR, DIR_RL, DIR_TB, EXPORTS, F32, IMPL_AUTO, IMPL_CHAIN, IMPL_FLAT, IMPL_FUSED, IMPL_NAIVE, IMPL_PAIR, IMPL_PLANE, IMPL_LINE,
    LIB_PATH, GspnError, gspn_last_launch_count, gspn_last_variant, gspn_merge, gspn_normalize_bwd, gspn_normalize_fwd, gspn_scan_bwd, gspn_scan_fwd_bwd_host,
    gspn_scan_bwd_host, gspn_scan_fwd, gspn_scan_fwd_host, gspn_version, lib,
)
