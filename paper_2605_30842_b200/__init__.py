"""paper_2605_30842_b200 — B200-native paged decode attention (CoMem's decode hot path).

The product is the C-ABI library built from ``csrc/`` (``include/comem_decode_attn.h``);
this package is its thin Python binding plus the seeded input generators
(``workloads``).  Importing the package does not load the library; the first
call does, and raises if it has not been built (no CPU fallback exists).
"""
from .binding import (  # noqa: F401
    COMEM_ERR_CUDA,
    COMEM_ERR_INVALID_ARG,
    COMEM_ERR_UNSUPPORTED,
    COMEM_ERR_WORKSPACE,
    COMEM_OK,
    ComemError,
    alloc_workspace,
    comem_decode_attn,
    comem_decode_attn_async,
    comem_decode_attn_phases_async,
    comem_decode_attn_window_async,
    COMEM_PHASE_SPLIT,
    COMEM_PHASE_COMBINE,
    comem_decode_attn_fp8_async,
    comem_prefill_attn_async,
    comem_decode_attn_workspace_bytes,
    comem_decode_saving_seconds,
    comem_kstep_context_lengths,
    comem_kstep_plan,
    comem_max_compression_ratio,
    comem_net_speedup,
    comem_decode_step_host,
    comem_grid_ctas,
    comem_kv_append_async,
    comem_kv_append_fp8_async,
    comem_schedule_host,
    comem_set_grid_ctas,
    comem_sm_partition,
    comem_read_ceiling_async,
    COMEM_READ_CEILING_SINK_WORDS,
    LaunchOpts,
    comem_set_programmatic_launch,
    comem_validate_inputs,
    comem_status_string,
    comem_version,
    comem_workspace_init_async,
    library_path,
    load_library,
)
