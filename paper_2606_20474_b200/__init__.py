"""paper_2606_20474_b200 — B200-native UltraQuant KV-cache hot path (arxiv/paper_2606_20474).

Thin Python binding over the C-ABI CUDA library libuq.so (include/uq.h): argument marshalling
only — every step of the path (rotation, quantiser, paged split-K attention, merge) runs in the
hand-written sm_100a kernels under csrc/.  PyTorch is used for device memory and streams.

There is NO CPU fallback: if libuq.so is missing or does not load, every entry point raises.
"""
from .binding import (  # noqa: F401
    UQConfig,
    UQError,
    RECORD_BYTES,
    record_bytes,
    StepBuffers,
    StepGraph,
    HostStage,
    HostStepGraph,
    alloc_cache,
    alloc_baseline_cache,
    baseline_append,
    baseline_decode_attention,
    baseline_decode_step,
    baseline_record_bytes,
    KV_BF16,
    KV_FP8_E4M3,
    KV_ULTRA_TQ,
    tq_append,
    tq_decode_attention,
    cache_record_bytes,
    calibrate_c,
    PrefixBuffers,
    decode_attention,
    decode_attention_shared_prefix,
    decode_attention_static,
    decode_static_scratch_needed,
    static_scratch_bytes,
    decode_step,
    decode_step_host,
    decode_workspace_bytes,
    FLAG_DEBUG_CHECKS,
    FLAG_NO_BULK_APPEND,
    FLAG_SMALL_APPEND_AHEAD,
    last_error,
    library_path,
    merge_splits,
    rotate_quantize_append,
    suggest_num_splits,
    suggest_prefix_splits,
    suggest_num_splits_max,
)
