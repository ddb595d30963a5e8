"""Convenience wrappers over the C-ABI calls: allocate with torch, marshal, launch.

No arithmetic of the method happens here -- layout, pack, attention and combine all run in
libupr's kernels.  PyTorch provides device memory and the stream only.
"""
from __future__ import annotations

import dataclasses
from typing import Optional

import numpy as np
import torch

from . import binding as B_

_TORCH_DT = {B_.UPR_F32: torch.float32, B_.UPR_BF16: torch.bfloat16}
DTYPE_ID = {"f32": B_.UPR_F32, "bf16": B_.UPR_BF16, "fp8": B_.UPR_FP8_E4M3}


@dataclasses.dataclass
class DecodeCache:
    """The ranking consumer's packed decode cache for one batch of users."""
    layout: B_.KvLayout
    row_off: np.ndarray            # host int64 [B+1]
    k_cache: torch.Tensor          # uint8 [bytes_cache]
    v_cache: torch.Tensor
    k_scale: Optional[torch.Tensor]  # fp32 [n_layers*H] (FP8) or None
    v_scale: Optional[torch.Tensor]
    seq_lens: torch.Tensor         # device int32 [B]
    max_seq_len: int


def alloc_cache(seq_lens_host, H: int, d: int, n_layers: int, kv_dtype: int, device) -> DecodeCache:
    lay, row_off = B_.upr_kv_cache_layout(seq_lens_host, H, d, n_layers, kv_dtype)
    k = torch.empty(lay.bytes_cache, dtype=torch.uint8, device=device)
    v = torch.empty(lay.bytes_cache, dtype=torch.uint8, device=device)
    ks = vs = None
    if kv_dtype == B_.UPR_FP8_E4M3:
        ks = torch.empty(n_layers * H, dtype=torch.float32, device=device)
        vs = torch.empty(n_layers * H, dtype=torch.float32, device=device)
    sl = torch.as_tensor(np.asarray(seq_lens_host, dtype=np.int32), device=device)
    mx = int(np.max(seq_lens_host)) if len(seq_lens_host) else 0
    return DecodeCache(lay, row_off, k, v, ks, vs, sl, mx)


def pack_cache(cache: DecodeCache, k_pool: torch.Tensor, v_pool: torch.Tensor, slot_ids: torch.Tensor,
               stream=None) -> DecodeCache:
    """a1: pool slots -> packed decode cache (upr_kv_pack)."""
    B_.upr_kv_pack(k_pool, v_pool, slot_ids, cache.seq_lens, cache.layout, cache.k_cache, cache.v_cache,
                   cache.k_scale, cache.v_scale, stream)
    return cache


class CrossAttention:
    """a2-a8 for a fixed problem shape: owns the output and workspace buffers."""

    def __init__(self, cache: DecodeCache, cand_offsets_host, q_dtype: int = B_.UPR_BF16, num_splits: int = 0,
                 device=None):
        lay = cache.layout
        self.cache = cache
        self.B, self.H, self.d, self.n_layers = lay.B, lay.H, lay.d, lay.n_layers
        self.q_dtype = q_dtype
        co = np.asarray(cand_offsets_host, dtype=np.int32)
        self.total_q = int(co[-1])
        device = device or cache.k_cache.device
        self.cand_offsets = torch.as_tensor(co, device=device)
        self.num_splits = num_splits
        self.splits = B_.upr_cross_attn_num_splits(self.B, self.H, self.d, self.n_layers, self.total_q, num_splits,
                                                   cache.max_seq_len)
        nbytes = B_.upr_cross_attn_workspace_bytes(self.B, self.H, self.d, self.n_layers, self.total_q, num_splits,
                                                   cache.max_seq_len)
        self.workspace = torch.empty(max(nbytes, 256), dtype=torch.uint8, device=device)
        self.out = torch.empty((self.n_layers, self.total_q, self.H, self.d), dtype=torch.float32, device=device)

    def __call__(self, q, k_self=None, v_self=None, sm_scale: float = 0.0, stream=None) -> torch.Tensor:
        c = self.cache
        B_.upr_cross_attn_fwd_ex(q, c.k_cache, c.v_cache, c.seq_lens, self.cand_offsets, self.out, self.B, self.H,
                                 self.d, self.n_layers, c.layout.dtype, self.q_dtype, self.total_q, self.workspace,
                                 k_self, v_self, c.k_scale, c.v_scale, sm_scale, self.num_splits, c.max_seq_len,
                                 stream)
        return self.out
