"""ctypes binding of libupr.so: same names as include/upr.h, argument marshalling only."""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import numpy as np
import torch

UPR_F32, UPR_BF16, UPR_FP8_E4M3, UPR_FP8_E4M3_USER = 0, 1, 2, 3
UPR_KV_PACKED, UPR_KV_POOL = 0, 1
UPR_KERNEL_AUTO, UPR_KERNEL_SINGLE, UPR_KERNEL_PAIR = 0, 1, 2
UPR_ROW_ALIGN, UPR_TAIL_ROWS = 16, 128
EXPORTED_SYMBOLS = [
    "upr_kv_cache_layout", "upr_kv_pack", "upr_cross_attn_fwd", "upr_cross_attn_fwd_ex", "upr_cross_attn_fwd_noalloc", "upr_cross_attn_noalloc_scratch_bytes",
    "upr_cross_attn_workspace_bytes", "upr_cross_attn_num_splits", "upr_last_launch_count",
    "upr_last_error", "upr_version", "upr_last_attn_kernel", "upr_linear_fp8_ex_fwd", "upr_layernorm_fp8_fwd",
    "upr_linear_fwd", "upr_linear_residual_fwd", "upr_linear_fp8_fwd", "upr_layernorm_fwd", "upr_kv_project_into_pool", "upr_action_utility", "upr_topk_per_user",
    "upr_pool_export", "upr_pool_open", "upr_pool_close", "upr_slot_ring_init", "upr_slot_ring_acquire",
]
UPR_ACT_NONE, UPR_ACT_SILU, UPR_ACT_RELU = 0, 1, 2
UPR_IPC_HANDLE_BYTES = 80

_HERE = os.path.dirname(os.path.abspath(__file__))


def lib_path() -> str:
    return os.path.join(_HERE, "libupr.so")


class UprError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"libupr status {status}: {msg}")
        self.status = status


class KvLayout(ctypes.Structure):
    _fields_ = [
        ("B", ctypes.c_int32), ("H", ctypes.c_int32), ("d", ctypes.c_int32), ("n_layers", ctypes.c_int32),
        ("dtype", ctypes.c_int32), ("row_align", ctypes.c_int32), ("tail_rows", ctypes.c_int32),
        ("elem_bytes", ctypes.c_int32), ("R", ctypes.c_int64), ("row_bytes", ctypes.c_int64),
        ("head_stride_bytes", ctypes.c_int64), ("layer_stride_bytes", ctypes.c_int64),
        ("bytes_cache", ctypes.c_int64), ("bytes_scales", ctypes.c_int64),
    ]


class _AttnParams(ctypes.Structure):
    _fields_ = [
        ("q", ctypes.c_void_p), ("k_cache", ctypes.c_void_p), ("v_cache", ctypes.c_void_p),
        ("seq_lens", ctypes.c_void_p), ("cand_offsets", ctypes.c_void_p), ("out", ctypes.c_void_p),
        ("k_self", ctypes.c_void_p), ("v_self", ctypes.c_void_p),
        ("k_scale", ctypes.c_void_p), ("v_scale", ctypes.c_void_p),
        ("B", ctypes.c_int32), ("H", ctypes.c_int32), ("d", ctypes.c_int32), ("n_layers", ctypes.c_int32),
        ("kv_dtype", ctypes.c_int32), ("q_dtype", ctypes.c_int32),
        ("total_q", ctypes.c_int64), ("sm_scale", ctypes.c_float), ("num_splits", ctypes.c_int32),
        ("max_seq_len", ctypes.c_int32), ("workspace", ctypes.c_void_p), ("workspace_bytes", ctypes.c_size_t),
        ("kv_source", ctypes.c_int32), ("pool_slots", ctypes.c_int32), ("pool_n_max", ctypes.c_int32),
        ("H_kv", ctypes.c_int32), ("slot_ids", ctypes.c_void_p), ("kv_bytes", ctypes.c_int64),
        ("kv_rows", ctypes.c_int64), ("causal", ctypes.c_int32), ("kernel", ctypes.c_int32),
    ]


_lib: Optional[ctypes.CDLL] = None


def _load() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        path = lib_path()
        if not os.path.exists(path):
            raise ImportError(
                f"{path} is missing: build it with `python -m paper_2606_00422_b200.build` "
                "(nvcc, sm_100a). There is no CPU fallback.")
        lib = ctypes.CDLL(path)
        lib.upr_last_error.restype = ctypes.c_char_p
        lib.upr_version.restype = ctypes.c_char_p
        lib.upr_last_launch_count.restype = ctypes.c_int
        lib.upr_last_attn_kernel.restype = ctypes.c_char_p
        lib.upr_cross_attn_workspace_bytes.restype = ctypes.c_size_t
        lib.upr_cross_attn_workspace_bytes.argtypes = [ctypes.POINTER(_AttnParams)]
        lib.upr_cross_attn_num_splits.restype = ctypes.c_int
        lib.upr_cross_attn_num_splits.argtypes = [ctypes.POINTER(_AttnParams)]
        lib.upr_kv_cache_layout.restype = ctypes.c_int
        lib.upr_kv_cache_layout.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                            ctypes.c_int, ctypes.POINTER(KvLayout), ctypes.c_void_p]
        lib.upr_kv_pack.restype = ctypes.c_int
        lib.upr_kv_pack.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_void_p,
                                    ctypes.c_void_p, ctypes.POINTER(KvLayout), ctypes.c_void_p, ctypes.c_void_p,
                                    ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        lib.upr_cross_attn_fwd.restype = ctypes.c_int
        lib.upr_cross_attn_fwd.argtypes = [ctypes.c_void_p] * 6 + [ctypes.c_int] * 4 + [ctypes.c_void_p]
        lib.upr_cross_attn_fwd_noalloc.restype = ctypes.c_int
        lib.upr_cross_attn_fwd_noalloc.argtypes = [ctypes.POINTER(_AttnParams), ctypes.c_void_p]
        lib.upr_cross_attn_noalloc_scratch_bytes.restype = ctypes.c_size_t
        lib.upr_cross_attn_noalloc_scratch_bytes.argtypes = []
        lib.upr_cross_attn_fwd_ex.restype = ctypes.c_int
        lib.upr_cross_attn_fwd_ex.argtypes = [ctypes.POINTER(_AttnParams), ctypes.c_void_p]
        lib.upr_linear_fwd.restype = ctypes.c_int
        lib.upr_linear_fwd.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
                                       ctypes.c_int, ctypes.c_int64, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                       ctypes.c_void_p]
        lib.upr_linear_residual_fwd.restype = ctypes.c_int
        lib.upr_linear_residual_fwd.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p,
                                                ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_int,
                                                ctypes.c_int, ctypes.c_int, ctypes.c_void_p]
        lib.upr_linear_fp8_fwd.restype = ctypes.c_int
        lib.upr_linear_fp8_fwd.argtypes = [ctypes.c_void_p, ctypes.c_float, ctypes.c_void_p, ctypes.c_float, ctypes.c_void_p,
                                           ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_int,
                                           ctypes.c_int, ctypes.c_int, ctypes.c_void_p]
        lib.upr_linear_fp8_ex_fwd.restype = ctypes.c_int
        lib.upr_linear_fp8_ex_fwd.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_float, ctypes.c_void_p, ctypes.c_float,
                                              ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int,
                                              ctypes.c_float, ctypes.c_int64, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                              ctypes.c_void_p]
        lib.upr_layernorm_fwd.restype = ctypes.c_int
        lib.upr_layernorm_fwd.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64,
                                          ctypes.c_int, ctypes.c_float, ctypes.c_void_p]
        lib.upr_layernorm_fp8_fwd.restype = ctypes.c_int
        lib.upr_layernorm_fp8_fwd.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_float,
                                              ctypes.c_int64, ctypes.c_int, ctypes.c_float, ctypes.c_void_p]
        lib.upr_kv_project_into_pool.restype = ctypes.c_int
        lib.upr_kv_project_into_pool.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p,
                                                 ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64] + \
                                                [ctypes.c_int] * 7 + [ctypes.c_void_p]
        lib.upr_action_utility.restype = ctypes.c_int
        lib.upr_action_utility.argtypes = [ctypes.c_void_p] * 4 + [ctypes.c_int64, ctypes.c_int, ctypes.c_int,
                                                                   ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        lib.upr_topk_per_user.restype = ctypes.c_int
        lib.upr_topk_per_user.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                          ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        lib.upr_pool_export.restype = ctypes.c_int
        lib.upr_pool_export.argtypes = [ctypes.c_void_p, ctypes.c_void_p]
        lib.upr_pool_open.restype = ctypes.c_int
        lib.upr_pool_open.argtypes = [ctypes.c_void_p, ctypes.POINTER(ctypes.c_void_p)]
        lib.upr_pool_close.restype = ctypes.c_int
        lib.upr_pool_close.argtypes = [ctypes.c_void_p]
        lib.upr_slot_ring_init.restype = ctypes.c_int
        lib.upr_slot_ring_init.argtypes = [ctypes.c_void_p, ctypes.c_int32]
        lib.upr_slot_ring_acquire.restype = ctypes.c_int
        lib.upr_slot_ring_acquire.argtypes = [ctypes.c_void_p, ctypes.c_int32, ctypes.c_void_p]
        _lib = lib
    return _lib


def _check(status: int) -> None:
    if status != 0:
        raise UprError(status, _load().upr_last_error().decode())


def _ptr(t: Optional[torch.Tensor]) -> Optional[int]:
    if t is None:
        return None
    assert t.is_contiguous(), "libupr takes contiguous tensors"
    return t.data_ptr()


def _stream(stream) -> Optional[int]:
    if stream is None:
        stream = torch.cuda.current_stream()
    return stream.cuda_stream or None


def upr_version() -> str:
    return _load().upr_version().decode()


def upr_last_attn_kernel() -> str:
    return _load().upr_last_attn_kernel().decode()


def upr_last_launch_count() -> int:
    return int(_load().upr_last_launch_count())


def upr_kv_cache_layout(seq_lens, H: int, d: int, n_layers: int, dtype: int):
    """Host-only. seq_lens: host int32 array-like [B]. Returns (KvLayout, row_off int64 [B+1])."""
    sl = np.ascontiguousarray(np.asarray(seq_lens, dtype=np.int32))
    B = int(sl.shape[0])
    lay = KvLayout()
    row_off = np.zeros(B + 1, dtype=np.int64)
    _check(_load().upr_kv_cache_layout(sl.ctypes.data, B, H, d, n_layers, dtype, ctypes.byref(lay),
                                       row_off.ctypes.data))
    return lay, row_off


def upr_kv_pack(k_pool, v_pool, slot_ids, seq_lens, layout: KvLayout, k_cache, v_cache,
                k_scale=None, v_scale=None, stream=None) -> None:
    """Pools: device bf16 [n_layers, S, H, n_max, d]; slot_ids/seq_lens: device int32 [B]."""
    ref = k_pool if k_pool is not None else v_pool
    S, n_max = int(ref.shape[1]), int(ref.shape[3])
    _check(_load().upr_kv_pack(_ptr(k_pool), _ptr(v_pool), S, n_max, _ptr(slot_ids), _ptr(seq_lens),
                               ctypes.byref(layout), _ptr(k_cache), _ptr(v_cache), _ptr(k_scale), _ptr(v_scale),
                               _stream(stream)))


def upr_cross_attn_fwd(q, k_cache, v_cache, seq_lens, cand_offsets, out, B: int, H: int, d: int, dtype: int,
                       stream=None) -> None:
    _check(_load().upr_cross_attn_fwd(_ptr(q), _ptr(k_cache), _ptr(v_cache), _ptr(seq_lens), _ptr(cand_offsets),
                                      _ptr(out), B, H, d, dtype, _stream(stream)))


def _params(q, k_cache, v_cache, seq_lens, cand_offsets, out, B, H, d, n_layers, kv_dtype, q_dtype, total_q,
            k_self=None, v_self=None, k_scale=None, v_scale=None, sm_scale=0.0, num_splits=0, max_seq_len=0,
            workspace=None, kv_source=UPR_KV_PACKED, pool_slots=0, pool_n_max=0, H_kv=0, slot_ids=None,
            kv_bytes=0, kv_rows=0, kernel=UPR_KERNEL_AUTO, causal=0) -> _AttnParams:
    p = _AttnParams()
    p.q, p.k_cache, p.v_cache = _ptr(q), _ptr(k_cache), _ptr(v_cache)
    p.seq_lens, p.cand_offsets, p.out = _ptr(seq_lens), _ptr(cand_offsets), _ptr(out)
    p.k_self, p.v_self, p.k_scale, p.v_scale = _ptr(k_self), _ptr(v_self), _ptr(k_scale), _ptr(v_scale)
    p.B, p.H, p.d, p.n_layers, p.kv_dtype, p.q_dtype = B, H, d, n_layers, kv_dtype, q_dtype
    p.total_q, p.sm_scale, p.num_splits, p.max_seq_len = total_q, sm_scale, num_splits, max_seq_len
    p.workspace = _ptr(workspace)
    p.workspace_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
    p.kv_source, p.pool_slots, p.pool_n_max, p.H_kv = kv_source, pool_slots, pool_n_max, H_kv
    p.slot_ids, p.kv_bytes, p.kv_rows, p.kernel, p.causal = _ptr(slot_ids), kv_bytes, kv_rows, kernel, int(causal)
    return p


def upr_cross_attn_workspace_bytes(B, H, d, n_layers, total_q, num_splits=0, max_seq_len=0, H_kv=0,
                                   kv_dtype=UPR_BF16, q_dtype=UPR_BF16, kernel=UPR_KERNEL_AUTO, causal=0) -> int:
    p = _params(None, None, None, None, None, None, B, H, d, n_layers, kv_dtype, q_dtype, total_q,
                num_splits=num_splits, max_seq_len=max_seq_len, H_kv=H_kv, kernel=kernel, causal=causal)
    return int(_load().upr_cross_attn_workspace_bytes(ctypes.byref(p)))


def upr_cross_attn_num_splits(B, H, d, n_layers, total_q, num_splits=0, max_seq_len=0, H_kv=0,
                              kv_dtype=UPR_BF16, q_dtype=UPR_BF16, kernel=UPR_KERNEL_AUTO, causal=0) -> int:
    p = _params(None, None, None, None, None, None, B, H, d, n_layers, kv_dtype, q_dtype, total_q,
                num_splits=num_splits, max_seq_len=max_seq_len, H_kv=H_kv, kernel=kernel, causal=causal)
    return int(_load().upr_cross_attn_num_splits(ctypes.byref(p)))


def upr_cross_attn_fwd_ex(q, k_cache, v_cache, seq_lens, cand_offsets, out, B, H, d, n_layers, kv_dtype, q_dtype,
                          total_q, workspace, k_self=None, v_self=None, k_scale=None, v_scale=None, sm_scale=0.0,
                          num_splits=0, max_seq_len=0, stream=None, kv_source=UPR_KV_PACKED, pool_slots=0,
                          pool_n_max=0, H_kv=0, slot_ids=None, kv_bytes=0, kv_rows=0,
                          kernel=UPR_KERNEL_AUTO, causal=0) -> None:
    """k_cache / v_cache are packed decode caches, or (kv_source=UPR_KV_POOL) the bf16 pools
    [n_layers, pool_slots, H_kv, pool_n_max, d] read in place through slot_ids."""
    p = _params(q, k_cache, v_cache, seq_lens, cand_offsets, out, B, H, d, n_layers, kv_dtype, q_dtype, total_q,
                k_self, v_self, k_scale, v_scale, sm_scale, num_splits, max_seq_len, workspace, kv_source,
                pool_slots, pool_n_max, H_kv, slot_ids, kv_bytes, kv_rows, kernel, causal)
    _check(_load().upr_cross_attn_fwd_ex(ctypes.byref(p), _stream(stream)))


def upr_cross_attn_fwd_noalloc(q, k_cache, v_cache, seq_lens, cand_offsets, out, B, H, d, n_layers, kv_dtype, q_dtype,
                               total_q, k_self=None, v_self=None, k_scale=None, v_scale=None, sm_scale=0.0,
                               num_splits=0, max_seq_len=0, stream=None, kv_source=UPR_KV_PACKED, pool_slots=0,
                               pool_n_max=0, H_kv=0, slot_ids=None, kv_bytes=0, kv_rows=0,
                               kernel=UPR_KERNEL_AUTO, causal=0) -> None:
    """upr_cross_attn_fwd_ex without a workspace argument: the scratch is a static device array in the library
    (upr_cross_attn_noalloc_scratch_bytes() long); no allocation happens in the call."""
    p = _params(q, k_cache, v_cache, seq_lens, cand_offsets, out, B, H, d, n_layers, kv_dtype, q_dtype, total_q,
                k_self, v_self, k_scale, v_scale, sm_scale, num_splits, max_seq_len, None, kv_source,
                pool_slots, pool_n_max, H_kv, slot_ids, kv_bytes, kv_rows, kernel, causal)
    _check(_load().upr_cross_attn_fwd_noalloc(ctypes.byref(p), _stream(stream)))


def upr_cross_attn_noalloc_scratch_bytes() -> int:
    return int(_load().upr_cross_attn_noalloc_scratch_bytes())


# ---------------------------------------------------------------------------- decode-layer tail, consumer, pool
_DT = {torch.float32: UPR_F32, torch.bfloat16: UPR_BF16}


def upr_linear_fwd(x, w, bias, y, act: int = UPR_ACT_NONE, stream=None) -> None:
    """y = act(x W^T + bias): x [M,K] bf16/fp32, w [N,K] bf16, bias fp32 [N] or None, y [M,N] bf16/fp32."""
    M, K = int(x.shape[0]), int(x.shape[1])
    N = int(w.shape[0])
    _check(_load().upr_linear_fwd(_ptr(x), _DT[x.dtype], _ptr(w), _ptr(bias), _ptr(y), _DT[y.dtype], M, N, K, act,
                                  _stream(stream)))


def upr_linear_residual_fwd(x, w, bias, residual, y, act: int = UPR_ACT_NONE, stream=None) -> None:
    """y = act(x W^T + bias) + residual (bf16 [M,N], may alias y)."""
    M, K = int(x.shape[0]), int(x.shape[1])
    N = int(w.shape[0])
    _check(_load().upr_linear_residual_fwd(_ptr(x), _DT[x.dtype], _ptr(w), _ptr(bias), _ptr(residual), _ptr(y),
                                           _DT[y.dtype], M, N, K, act, _stream(stream)))


def upr_linear_fp8_fwd(x, x_scale: float, w8, w_scale: float, bias, residual, y, act: int = UPR_ACT_NONE,
                       stream=None) -> None:
    """FP8 E4M3 linear: x bf16 [M,K] quantised in-kernel with x_scale, w8 uint8 E4M3 bytes [N,K] with w_scale."""
    M, K = int(x.shape[0]), int(x.shape[1])
    N = int(w8.shape[0])
    _check(_load().upr_linear_fp8_fwd(_ptr(x), x_scale, _ptr(w8), w_scale, _ptr(bias), _ptr(residual), _ptr(y),
                                      _DT[y.dtype], M, N, K, act, _stream(stream)))


def upr_linear_fp8_ex_fwd(x, x_scale: float, w8, w_scale: float, bias, residual, y, y_scale: float = 1.0,
                          act: int = UPR_ACT_NONE, stream=None) -> None:
    """FP8 E4M3 linear inside a chain: x bf16 [M,K] (quantised in-kernel) or uint8 E4M3 bytes; y bf16 / fp32 or
    uint8 E4M3 bytes (quantised with y_scale)."""
    M, K = int(x.shape[0]), int(x.shape[1])
    N = int(w8.shape[0])
    xd = UPR_FP8_E4M3 if x.dtype == torch.uint8 else _DT[x.dtype]
    yd = UPR_FP8_E4M3 if y.dtype == torch.uint8 else _DT[y.dtype]
    _check(_load().upr_linear_fp8_ex_fwd(_ptr(x), xd, x_scale, _ptr(w8), w_scale, _ptr(bias), _ptr(residual), _ptr(y),
                                         yd, y_scale, M, N, K, act, _stream(stream)))


def upr_layernorm_fwd(x, gamma, beta, y, eps: float = 1e-5, stream=None) -> None:
    """x, y bf16 [M, D]; gamma, beta fp32 [D]."""
    _check(_load().upr_layernorm_fwd(_ptr(x), _ptr(gamma), _ptr(beta), _ptr(y), int(x.shape[0]), int(x.shape[1]), eps,
                                     _stream(stream)))


def upr_layernorm_fp8_fwd(x, gamma, beta, y8, y_scale: float, eps: float = 1e-5, stream=None) -> None:
    """x bf16 [M, D]; y8 uint8 E4M3 bytes [M, D] quantised with y_scale; gamma, beta fp32 [D]."""
    _check(_load().upr_layernorm_fp8_fwd(_ptr(x), _ptr(gamma), _ptr(beta), _ptr(y8), y_scale, int(x.shape[0]),
                                         int(x.shape[1]), eps, _stream(stream)))


def upr_kv_project_into_pool(x, w, bias, pool, tok_slot, tok_pos, layer: int, stream=None) -> None:
    """pool[layer, tok_slot[m], h, tok_pos[m], :] = (x[m] W^T + bias)[h*d:(h+1)*d]; pool bf16 [layers,S,H,n,d]."""
    n_layers, S, H, n, d = (int(v) for v in pool.shape)
    M, K = int(x.shape[0]), int(x.shape[1])
    assert int(w.shape[0]) == H * d and int(w.shape[1]) == K and pool.dtype == torch.bfloat16
    _check(_load().upr_kv_project_into_pool(_ptr(x), _DT[x.dtype], _ptr(w), _ptr(bias), _ptr(pool), _ptr(tok_slot),
                                            _ptr(tok_pos), M, K, layer, n_layers, S, H, n, d, _stream(stream)))


def upr_action_utility(hid, w2, b2, wc, probs, util, stream=None) -> None:
    """hid bf16 [M, C*Dh]; w2 fp32 [C,Dh]; b2, wc fp32 [C]; probs fp32 [M,C] or None; util fp32 [M]."""
    C, Dh = int(w2.shape[0]), int(w2.shape[1])
    M = int(hid.shape[0])
    _check(_load().upr_action_utility(_ptr(hid), _ptr(w2), _ptr(b2), _ptr(wc), M, C, Dh, _ptr(probs), _ptr(util),
                                      _stream(stream)))


def upr_topk_per_user(util, cand_offsets, K: int, max_cands: int, out_idx, out_cnt, stream=None) -> None:
    B = int(cand_offsets.shape[0]) - 1
    _check(_load().upr_topk_per_user(_ptr(util), _ptr(cand_offsets), B, K, max_cands, _ptr(out_idx), _ptr(out_cnt),
                                     _stream(stream)))


def upr_pool_export(pool: torch.Tensor) -> bytes:
    """Opaque handle bytes for the device memory of `pool`: CUDA IPC handle + offset."""
    buf = (ctypes.c_ubyte * UPR_IPC_HANDLE_BYTES)()
    _check(_load().upr_pool_export(pool.data_ptr(), ctypes.byref(buf)))
    return bytes(buf)


def upr_pool_open(handle: bytes) -> int:
    """Map the exporter's allocation into this process; returns the device pointer."""
    buf = (ctypes.c_ubyte * UPR_IPC_HANDLE_BYTES).from_buffer_copy(handle)
    out = ctypes.c_void_p()
    _check(_load().upr_pool_open(ctypes.byref(buf), ctypes.byref(out)))
    return int(out.value)


def upr_pool_close(ptr: int) -> None:
    _check(_load().upr_pool_close(ctypes.c_void_p(ptr)))


class SlotRing(ctypes.Structure):
    """Round-robin slot assignment."""
    _fields_ = [("S", ctypes.c_int32), ("next", ctypes.c_int32)]

    def __init__(self, S: int):
        super().__init__()
        _check(_load().upr_slot_ring_init(ctypes.byref(self), S))

    def acquire(self, n: int) -> np.ndarray:
        out = np.zeros(n, dtype=np.int32)
        _check(_load().upr_slot_ring_acquire(ctypes.byref(self), n, out.ctypes.data))
        return out
