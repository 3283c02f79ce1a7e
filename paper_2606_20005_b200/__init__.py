"""paper_2606_20005_b200 -- B200-native StreamKL (fused attention-KL forward/backward, arxiv/paper_2606_20005).

The product is the C-ABI library `libstreamkl.so` (declared in include/streamkl.h, built from csrc/ for
sm_100a).  This package is the thin Python binding: argument marshalling only, every step of the hot path
runs in the CUDA kernels.  There is no CPU fallback -- importing the binding without the built library raises.
"""
from .binding import (  # noqa: F401
    StreamKLError,
    lib,
    lib_path,
    streamkl_bwd,
    streamkl_bwd_workspace_bytes,
    streamkl_fwd,
    streamkl_fwd_bwd_host,
    streamkl_fwd_host,
    streamkl_fwd_splitk,
    streamkl_fwd_splitk_noalloc,
    streamkl_fwd_splitk_noalloc_capacity,
    STREAMKL_ERR_SCRATCH_LIMIT,
    streamkl_host_trim,
    streamkl_set_bwd_mode,
    streamkl_set_fwd_plan,
    STREAMKL_FWD_SINGLE,
    STREAMKL_FWD_MULTICAST,
    STREAMKL_FWD_PAIR_MMA,
    STREAMKL_FWD_PERSISTENT,
    STREAMKL_FWD_PER_TILE,
    STREAMKL_FWD_AUTO,
    STREAMKL_BWD_AUTO,
    STREAMKL_BWD_SEPARATE,
    STREAMKL_BWD_FUSED,
    STREAMKL_BF16,
    STREAMKL_F16,
    STREAMKL_F32,
    StreamKLLayout,
    streamkl_fwd_splitk_splits,
    streamkl_fwd_splitk_workspace_bytes,
    streamkl_kernel_name,
    streamkl_last_launch_count,
    streamkl_profile_collect,
    streamkl_profile_enable,
    streamkl_strerror,
    streamkl_version,
)
