"""paper_2406_03243_b200 — B200-native live migration of a paged KV cache (Llumnix §4.2/§5).

Thin binding over the C-ABI library `libllx.so` (include/llx.h).  The functions here only
marshal arguments; every step of the path runs in the library's CUDA kernels.  Importing this
package needs the built library (`python -m paper_2406_03243_b200.build`); there is no CPU path.
"""
from .binding import (  # noqa: F401
    LlxError, Pool, lib, load, LaunchOpts, OPT_DEFAULT, ROUTE_AUTO, ROUTE_PEER, ROUTE_COPY_ENGINE,
    F16, BF16, U8,
    OPT_COPY_KERNEL, OPT_MAX_CTAS, OPT_CHUNK_BYTES, OPT_RING_STAGES, OPT_IDS_BY_VALUE_MAX, OPT_ATTN_SPLIT_TOKENS,
    OPT_UNIT_ORDER, OPT_L2_HINT, OPT_RINGS_PER_CTA, OPT_PDL, OPT_BANDWIDTH_GBPS, OPT_VIA_HOST_MODE, OPT_DYNAMIC_TAIL_PCT, OPT_DYNAMIC_TAIL_BATCH, OPT_EXACT_RESIDENCY, OPT_COPY_SMEM_CARVEOUT_PCT, OPT_PACED_SLICE_US, OPT_OVERLAP_PREV,
    pool_create, pool_wrap, pool_bytes_for, pool_ipc_export, pool_ipc_open, IPC_HANDLE_BYTES,
    plan_stage, predict_stage_sizes, migrate_stage, migrate_stage_wait, migrate_batch, staging_bytes, PinnedStaging, pack, unpack, migrate_via_host,
    append_tokens, decode_attention, decode_attention_static_ws, ATTN_STATIC_WS_BYTES,
    calc_freeness, pair_instances, migration_order, plan_migration_batch,
    BlockManager, Migration, BudgetController, REQ_RUNNING, REQ_FINISHED, REQ_PREEMPTED, REQ_PEER_FAILED,
    MIG_READY, MIG_COPYING, MIG_FINAL_COPYING, MIG_COMMITTED, MIG_ABORTED,
    ABORT_NONE, ABORT_FINISHED, ABORT_PREEMPTED, ABORT_PEER_FAILED, ABORT_NO_SPACE,
    set_option, get_option, options, synchronize, counters, reset_counters, version, EXPORTS,
)
