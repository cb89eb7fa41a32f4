"""paper_2606_04484_b200 — B200-native (sm_100a) timeline merging + policy-loss fwd/bwd.

The product is libajt.so (C ABI in include/ajt.h, CUDA sources in csrc/).  This package is a thin
argument-marshalling binding with the same names; every step of the path runs in the CUDA kernels.
There is no CPU fallback: calls raise if the CUDA library is missing or no device is present.
"""
from .binding import (  # noqa: F401
    AUTHOR_ENV,
    AUTHOR_LLM,
    AUTHOR_USER,
    AjtError,
    DT_BF16,
    DT_F32,
    MERGE_WEAK_HASH,
    OWNER_LONGEST,
    OWNER_PAPER,
    STATUS_BAD_OFFSETS,
    STATUS_BAD_SEG,
    STATUS_BAD_TARGET,
    STATUS_HASH_COLLISION,
    STATUS_INTERNAL,
    STATUS_PROBE_CAPACITY,
    STATUS_ZERO_LEN,
    exported_symbols,
    last_status,
    lib,
    library_path,
    lm_head_logp,
    loss_host_arena_bytes,
    loss_workspace_bytes,
    merge_blocks,
    merge_blocks_workspace_bytes,
    merge_host_arena_bytes,
    merge_timelines,
    merge_timelines_host,
    merge_workspace_bytes,
    pack_loss_inputs,
    policy_loss_fwd_bwd,
    policy_loss_fwd_bwd_ext,
    policy_loss_fwd_bwd_host,
    segment_counts,
    strerror,
    version,
)
