"""paper_1306_1392_b200 -- B200-native (sm_100a) projector pair, ramp filter and FBP of PyHST2.

The product is the C-ABI library declared in ``include/pyhst.h`` (hand-written CUDA under
``csrc/``); ``binding`` is a thin ctypes marshalling layer with the same names and
``workloads`` makes the seeded synthetic inputs.  There is no CPU fallback: every entry
point raises if the CUDA library is missing or no sm_100 device is present.
"""
from . import workloads  # noqa: F401
from .binding import (  # noqa: F401
    FILTER_RAMLAK, FILTER_SHEPP_LOGAN, FILTER_HANN, FILTER_HAMMING, FILTER_COSINE, SCAN_180, SCAN_360, SCAN_360_HALF, PyhstError,
    backproject, backproject_host, fbp, fbp_host, fista_tv, ista_tv, ring_filter, ring_filter_static, ecohe, cv_distance, patch_grid, patch_gradient, patch_fista, forward_project_host, forward_project, halfacq_extent, last_error, library_path, profile_enable, profile_read,
    ramp_filter, release_cache, set_backproject_variant, set_forward_project_variant, last_forward_project_kernel, set_halfacq_stitch, set_filter_variant, set_patch_gemm_variant, set_test_workspace_limit,
)
