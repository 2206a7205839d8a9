"""B200-native (sm_100a) Hierarchical Global Attention prefill hot path (arxiv/paper_2606_30709).

Thin ctypes binding over the C ABI in include/hga.h (libhga.so, hand-written CUDA).  The binding only marshals
arguments: every step of the path runs in the CUDA kernels.  There is no CPU fallback -- if libhga.so is missing or
no CUDA device is present, calls fail loudly.
"""
from .binding import (  # noqa: F401
    HgaError,
    HostPlan,
    Params,
    PrefillBuffers,
    RouteResult,
    hga_attend,
    hga_build_summaries,
    hga_default_n_hi,
    hga_n_hi_rule,
    hga_prefill,
    hga_prefill_profile,
    hga_prefill_window,
    hga_rope,
    hga_route,
    hga_route_static,
    hga_validate,
    hga_version,
    hga_workspace_bytes,
    lib_path,
    load_library,
    params_from_workload,
)
