"""paper_2606_17065_b200 -- B200-native (sm_100a) PIVOT implied-volatility hot path.

Thin Python binding over the C-ABI library `libpivot_iv.so` (include/pivot_iv.h).  Every step of the path runs in
the hand-written CUDA kernels; Python only marshals arguments.  PyTorch is used for device memory and streams.
There is no CPU fallback: calling any entry point without the built library or without a CUDA device raises.
"""
from .binding import (  # noqa: F401
    GATE_ATTENUATE,
    GATE_MASK,
    GATE_STRICT,
    RT_GATED,
    RT_NAIVE,
    FWD_AUTO,
    FWD_COMPACT,
    FWD_ROWWISE,
    FWD_FP64_ONLY,
    HOST_AUTO,
    HOST_STAGED,
    HOST_DIRECT,
    PivotError,
    Pipeline,
    ShardedPipeline,
    library_path,
    load_library,
    pivot_iv_black_price,
    pivot_iv_status_histogram,
    pivot_iv_backward,
    pivot_iv_backward_inputs,
    pivot_iv_forward,
    pivot_iv_forward_diag,
    pivot_iv_debug_math,
    pivot_iv_forward_ex,
    pivot_iv_forward_probe,
    pivot_iv_forward_host_static,
    STATIC_MAX_ROWS,
    pivot_iv_forward_launches,
    AUTO_MIN_ROWS,
    pivot_iv_forward_zones,
    pivot_iv_loss_price,
    pivot_iv_loss_roundtrip,
    pivot_iv_probe_dfma,
    pivot_iv_strerror,
    pivot_iv_version,
    EXPORTS,
)

__all__ = [
    "pivot_iv_forward", "pivot_iv_forward_zones", "pivot_iv_backward", "pivot_iv_backward_inputs", "pivot_iv_black_price", "pivot_iv_status_histogram",
    "pivot_iv_loss_price", "pivot_iv_loss_roundtrip",
    "Pipeline", "ShardedPipeline", "pivot_iv_probe_dfma",
    "pivot_iv_strerror", "pivot_iv_version", "load_library", "library_path", "PivotError", "GATE_MASK",
    "GATE_ATTENUATE", "GATE_STRICT", "RT_GATED", "RT_NAIVE", "FWD_AUTO", "FWD_COMPACT", "FWD_ROWWISE", "FWD_FP64_ONLY", "HOST_AUTO", "HOST_STAGED", "HOST_DIRECT", "pivot_iv_forward_ex", "pivot_iv_forward_diag", "pivot_iv_debug_math", "EXPORTS",
    "pivot_iv_forward_probe", "pivot_iv_forward_launches", "AUTO_MIN_ROWS",
    "pivot_iv_forward_host_static", "STATIC_MAX_ROWS",
]
