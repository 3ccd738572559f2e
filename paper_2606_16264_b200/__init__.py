"""tropical-b200: B200-native (sm_100a) hot path of one Tropical multiplexed iteration.

Thin Python binding over the C-ABI in include/tropical.h (argument marshalling only; every step
of the path runs in the library's CUDA kernels).  PyTorch is used for device memory and streams.
Importing this package never imports ``oracle``.
"""
from .binding import (  # noqa: F401
    Batch,
    CostBreakdown,
    CostModel,
    IterBreakdown,
    LayerShape,
    LinearModel,
    KVPool,
    SIM_COLOCATED,
    SIM_DISAGGREGATED,
    SIM_MULTIPLEXED,
    SimConfig,
    TIMELINE_FIELDS,
    TropicalError,
    debug_attention_simt,
    debug_read_profile,
    debug_set_grid,
    debug_timeline,
    debug_set_split_pages,
    debug_wait_profile,
    iter_cost,
    kv_append,
    kv_gather,
    kv_migrate,
    enable_peer_access,
    last_launch_count,
    lib,
    mixed_attention,
    sim_run,
    status_string,
    step_cost,
    validate_batch,
    step_host,
    step_host_staging_bytes,
    version,
    workspace_bytes,
)
