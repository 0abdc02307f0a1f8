"""libaffinescan for B200 (sm_100a): the affine-pair associative scan of
arxiv/paper_2606_00601 and the fused Mamba-style selective-scan forward.

The product is the C-ABI shared library (include/affinescan.h, csrc/); this package is
its thin ctypes binding.  There is no CPU fallback here, and nothing from the test-only CPU reference is imported.
"""
from .binding import (  # noqa: F401
    AFFINE_BLELLOCH,
    AFFINE_CTA_LOOP,
    AFFINE_LOOKBACK,
    AFFINE_WARP_SEQ,
    BF16,
    F32,
    OPT_LANE_ROW_G,
    OPT_LANE_ROW_POLY16,
    SELECTIVE_LANE_ROW,
    SELECTIVE_WARP_ROW,
    SELECTIVE_WARP_ROW_TMA,
    VARIANT_AUTO,
    VARIANT_NAMES,
    AffineScanError,
    affine_scan,
    affine_scan_ex,
    affine_scan_host,
    declared_symbols,
    last_cuda_error,
    last_variant,
    launch_count,
    library_path,
    load,
    release_cache,
    selective_scan_fwd,
    selective_scan_fwd_ex,
    selective_scan_fwd_host,
    set_option,
    status_string,
    version,
)
