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
DTYPE_ID = {"f32": B_.UPR_F32, "bf16": B_.UPR_BF16, "fp8": B_.UPR_FP8_E4M3, "fp8_user": B_.UPR_FP8_E4M3_USER}


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
    if lay.bytes_scales:
        ks = torch.empty(lay.bytes_scales // 4, dtype=torch.float32, device=device)
        vs = torch.empty(lay.bytes_scales // 4, dtype=torch.float32, device=device)
    sl = torch.as_tensor(np.asarray(seq_lens_host, dtype=np.int32), device=device)
    mx = int(np.max(seq_lens_host)) if len(seq_lens_host) else 0
    return DecodeCache(lay, row_off, k, v, ks, vs, sl, mx)


def pack_cache(cache: DecodeCache, k_pool: torch.Tensor, v_pool: torch.Tensor, slot_ids: torch.Tensor,
               stream=None) -> DecodeCache:
    """a1: pool slots -> packed decode cache (upr_kv_pack)."""
    B_.upr_kv_pack(k_pool, v_pool, slot_ids, cache.seq_lens, cache.layout, cache.k_cache, cache.v_cache,
                   cache.k_scale, cache.v_scale, stream)
    return cache


@dataclasses.dataclass
class PoolView:
    """The retrieval stage's KV pool ([L,S,H_kv,n,D] bf16) addressed IN PLACE for one
    batch of users: no slot copy (the copy PAPER.md:204 / 278 pays for)."""
    k_pool: torch.Tensor           # bf16 [n_layers, S, H_kv, n_max, d]
    v_pool: torch.Tensor
    slot_ids: torch.Tensor         # device int32 [B]
    seq_lens: torch.Tensor         # device int32 [B]
    max_seq_len: int

    @staticmethod
    def of(k_pool, v_pool, slot_ids, seq_lens_host) -> "PoolView":
        sl = torch.as_tensor(np.asarray(seq_lens_host, dtype=np.int32), device=k_pool.device)
        mx = int(np.max(seq_lens_host)) if len(seq_lens_host) else 0
        return PoolView(k_pool, v_pool, slot_ids, sl, mx)


class CrossAttention:
    """a2-a8 for a fixed problem shape: owns the output and workspace buffers."""

    def __init__(self, cache, cand_offsets_host, q_dtype: int = B_.UPR_BF16, num_splits: int = 0,
                 device=None, H_q: Optional[int] = None, kernel: int = B_.UPR_KERNEL_AUTO, causal: bool = False):
        """cache: a DecodeCache (packed) or a PoolView (zero copy).  H_q: query heads when they are a
        multiple of the KV heads (grouped queries); default = the KV head count."""
        self.cache = cache
        self.pool = isinstance(cache, PoolView)
        if self.pool:
            self.n_layers, S, self.H_kv, n_max, self.d = (int(x) for x in cache.k_pool.shape)
            self.B = int(cache.seq_lens.shape[0])
            self.kv_dtype = B_.UPR_BF16
            self.kv_kwargs = dict(kv_source=B_.UPR_KV_POOL, pool_slots=S, pool_n_max=n_max,
                                  slot_ids=cache.slot_ids,
                                  kv_bytes=cache.k_pool.numel() * cache.k_pool.element_size())
        else:
            lay = cache.layout
            self.B, self.H_kv, self.d, self.n_layers = lay.B, lay.H, lay.d, lay.n_layers
            self.kv_dtype = lay.dtype
            self.kv_kwargs = dict(kv_bytes=int(lay.bytes_cache), kv_rows=int(lay.R))
        self.H = H_q or self.H_kv
        self.kv_kwargs["H_kv"] = self.H_kv
        self.kv_kwargs["kernel"] = kernel
        self.kv_kwargs["causal"] = int(causal)
        self.q_dtype = q_dtype
        co = np.asarray(cand_offsets_host, dtype=np.int32)
        self.total_q = int(co[-1])
        device = device or cache.seq_lens.device
        self.cand_offsets = torch.as_tensor(co, device=device)
        self.num_splits = num_splits
        self.splits = B_.upr_cross_attn_num_splits(self.B, self.H, self.d, self.n_layers, self.total_q, num_splits,
                                                   cache.max_seq_len, self.H_kv, self.kv_dtype, q_dtype, kernel, int(causal))
        nbytes = B_.upr_cross_attn_workspace_bytes(self.B, self.H, self.d, self.n_layers, self.total_q, num_splits,
                                                   cache.max_seq_len, self.H_kv, self.kv_dtype, q_dtype, kernel, int(causal))
        self.workspace = torch.empty(max(nbytes, 256), dtype=torch.uint8, device=device)
        self.out = torch.empty((self.n_layers, self.total_q, self.H, self.d), dtype=torch.float32, device=device)

    def __call__(self, q, k_self=None, v_self=None, sm_scale: float = 0.0, stream=None) -> torch.Tensor:
        c = self.cache
        k, v = (c.k_pool, c.v_pool) if self.pool else (c.k_cache, c.v_cache)
        ks, vs = (None, None) if self.pool else (c.k_scale, c.v_scale)
        B_.upr_cross_attn_fwd_ex(q, k, v, c.seq_lens, self.cand_offsets, self.out, self.B, self.H,
                                 self.d, self.n_layers, self.kv_dtype, self.q_dtype, self.total_q, self.workspace,
                                 k_self, v_self, ks, vs, sm_scale, self.num_splits, c.max_seq_len,
                                 stream, **self.kv_kwargs)
        return self.out


class RankingDecodeLayer:
    """One pre-LN decoder layer of the candidate-only ranking pass (reading Q19), as a
    sequence of C-ABI calls -- no arithmetic here:
        h1 = LN1(x);  q, k_self, v_self = h1 Wq^T, h1 Wk^T, h1 Wv^T
        a  = cross-attention(q; cached history K/V of the user; own key/value)        (fp32)
        x2 = x + a Wo^T;  h2 = LN2(x2);  y = x2 + W2 silu(W1 h2 + b1) + b2
    x: bf16 [total_q, D]; weights bf16 [out, in] (synthetic), LN parameters fp32.  Buffers are allocated once.
    With `fp8_mlp` = {"w1_8", "w1_scale", "w2_8", "w2_scale", "h_scale", "u_scale"} (E4M3 weight bytes and per-tensor
    scales) the MLP runs as an FP8 chain: LN2 writes E4M3 bytes, both GEMMs take both operands as
    E4M3 through TMA, the hidden tensor stays E4M3 in between."""

    def __init__(self, attn: CrossAttention, D: int, hidden: int, params: dict, device=None, fp8_mlp: dict = None):
        self.attn = attn
        assert attn.n_layers == 1, "one attention object per layer"
        self.D, self.hidden, self.p = D, hidden, params
        M, Hq, Hkv, d = attn.total_q, attn.H, attn.H_kv, attn.d
        dev = device or attn.out.device
        bf = dict(dtype=torch.bfloat16, device=dev)
        self.h1 = torch.empty((M, D), **bf)
        self.q = torch.empty((1, M, Hq, d), **bf)
        self.ks = torch.empty((1, M, Hq, d), **bf)
        self.vs = torch.empty((1, M, Hq, d), **bf)
        self.x2 = torch.empty((M, D), **bf)
        self.h2 = torch.empty((M, D), **bf)
        self.u = torch.empty((M, hidden), **bf)
        self.y = torch.empty((M, D), **bf)
        self.fp8 = fp8_mlp
        if fp8_mlp is not None:
            self.h2_8 = torch.empty((M, D), dtype=torch.uint8, device=dev)
            self.u_8 = torch.empty((M, hidden), dtype=torch.uint8, device=dev)
        self.launches = 0

    def __call__(self, x: torch.Tensor, stream=None) -> torch.Tensor:
        p, a = self.p, self.attn
        M, Hq, d = a.total_q, a.H, a.d
        n = 0
        B_.upr_layernorm_fwd(x, p["ln1_g"], p["ln1_b"], self.h1, stream=stream); n += 1
        B_.upr_linear_fwd(self.h1, p["wq"], None, self.q.view(M, Hq * d), stream=stream); n += 1
        B_.upr_linear_fwd(self.h1, p["wk"], None, self.ks.view(M, Hq * d), stream=stream); n += 1
        B_.upr_linear_fwd(self.h1, p["wv"], None, self.vs.view(M, Hq * d), stream=stream); n += 1
        out = a(self.q, self.ks, self.vs, stream=stream); n += B_.upr_last_launch_count()
        B_.upr_linear_residual_fwd(out.view(M, Hq * d), p["wo"], None, x, self.x2, stream=stream); n += 1
        f8 = self.fp8
        if f8 is None:
            B_.upr_layernorm_fwd(self.x2, p["ln2_g"], p["ln2_b"], self.h2, stream=stream); n += 1
            B_.upr_linear_fwd(self.h2, p["w1"], p["b1"], self.u, B_.UPR_ACT_SILU, stream=stream); n += 1
            B_.upr_linear_residual_fwd(self.u, p["w2"], p["b2"], self.x2, self.y, stream=stream); n += 1
        else:
            B_.upr_layernorm_fp8_fwd(self.x2, p["ln2_g"], p["ln2_b"], self.h2_8, f8["h_scale"], stream=stream); n += 1
            B_.upr_linear_fp8_ex_fwd(self.h2_8, f8["h_scale"], f8["w1_8"], f8["w1_scale"], p["b1"], None, self.u_8,
                                     f8["u_scale"], B_.UPR_ACT_SILU, stream=stream); n += 1
            B_.upr_linear_fp8_ex_fwd(self.u_8, f8["u_scale"], f8["w2_8"], f8["w2_scale"], p["b2"], self.x2, self.y, 1.0,
                                     B_.UPR_ACT_NONE, stream=stream); n += 1
        self.launches = n
        return self.y
