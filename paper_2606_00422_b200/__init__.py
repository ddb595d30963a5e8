"""paper_2606_00422_b200 -- B200-native ranking cross-attention over a shared user-history KV
cache (the serving hot path of UniPinRec, arxiv/paper_2606_00422).

This package is a thin Python binding over the C-ABI library ``libupr.so`` (include/upr.h):
argument marshalling only; every step of the path runs in the CUDA kernels under ``csrc/``.
There is no CPU fallback: importing the binding fails loudly when the library is missing.
"""
from .binding import (  # noqa: F401
    UPR_BF16, UPR_F32, UPR_FP8_E4M3, UPR_FP8_E4M3_USER, UPR_KV_PACKED, UPR_KV_POOL, UPR_KERNEL_AUTO,
    UPR_KERNEL_SINGLE, UPR_KERNEL_PAIR, UPR_ROW_ALIGN, UPR_TAIL_ROWS, KvLayout, UprError, lib_path,
    upr_cross_attn_fwd, upr_cross_attn_fwd_ex, upr_cross_attn_fwd_noalloc, upr_cross_attn_noalloc_scratch_bytes, upr_cross_attn_num_splits, upr_cross_attn_workspace_bytes,
    upr_kv_cache_layout, upr_kv_pack, upr_last_attn_kernel, upr_linear_fwd, upr_linear_residual_fwd, upr_linear_fp8_fwd, upr_linear_fp8_ex_fwd, upr_layernorm_fwd, upr_layernorm_fp8_fwd, upr_kv_project_into_pool, upr_action_utility,
    upr_topk_per_user, upr_pool_export, upr_pool_open, upr_pool_close, SlotRing, UPR_ACT_NONE, UPR_ACT_SILU, UPR_ACT_RELU, upr_last_launch_count, upr_version, EXPORTED_SYMBOLS,
)
