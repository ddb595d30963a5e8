"""CPU fp64 oracle for the UniPinRec ranking cross-attention -- TEST INFRASTRUCTURE ONLY.

Thin ctypes binding over ``oracle/upr_oracle.c`` (plain C, fp64, the paper's definition
written out; see that file's header for citations and pins).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs
may import this package.  It imports nothing from ``paper_2606_00422_b200`` and the product
never imports it.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "upr_oracle.c")
_LIB = os.path.join(_HERE, "libupr_oracle.so")

F32, BF16, FP8_E4M3, FP8_E4M3_USER = 0, 1, 2, 3
ROW_ALIGN = 16  # DESIGN.md reading Q14


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no CUDA involved)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O3", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC", _SRC, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True, capture_output=True)
    return _LIB


_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.upro_bf16_to_f64.restype = ctypes.c_double
        _lib.upro_bf16_to_f64.argtypes = [ctypes.c_uint16]
        _lib.upro_f32_to_bf16.restype = ctypes.c_uint16
        _lib.upro_f32_to_bf16.argtypes = [ctypes.c_float]
        _lib.upro_e4m3_decode.restype = ctypes.c_double
        _lib.upro_e4m3_decode.argtypes = [ctypes.c_uint8]
        _lib.upro_e4m3_encode.restype = ctypes.c_uint8
        _lib.upro_e4m3_encode.argtypes = [ctypes.c_float]
        _lib.upro_num_threads.restype = ctypes.c_int
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _c64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads() -> int:
    return int(lib().upro_num_threads())


# ---------------------------------------------------------------------------- formats
def bf16_bits_to_f64(bits: np.ndarray) -> np.ndarray:
    """Exact widening of bfloat16 bit patterns (uint16) to float64."""
    bits = np.ascontiguousarray(bits, dtype=np.uint16)
    return (bits.astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.float32)
    f = lib().upro_f32_to_bf16
    return np.array([f(float(v)) for v in x.ravel()], dtype=np.uint16).reshape(x.shape)


def e4m3_decode(b: np.ndarray) -> np.ndarray:
    b = np.ascontiguousarray(b, dtype=np.uint8)
    f = lib().upro_e4m3_decode
    table = np.array([f(i) for i in range(256)], dtype=np.float64)
    return table[b]


def e4m3_encode(x: np.ndarray) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.float32)
    f = lib().upro_e4m3_encode
    return np.array([f(float(v)) for v in x.ravel()], dtype=np.uint8).reshape(x.shape)


# ---------------------------------------------------------------------------- layout
def layout(seq_lens, H: int, d: int, n_layers: int, dtype: int, align: int = ROW_ALIGN, tail_rows: int = 128):
    """Row-offset table and byte sizes of the packed cache (a0)."""
    seq_lens = np.ascontiguousarray(seq_lens, dtype=np.int32)
    B = int(seq_lens.shape[0])
    row_off = np.zeros(B + 1, dtype=np.int64)
    o7 = np.zeros(7, dtype=np.int64)
    rc = lib().upro_layout(_p(seq_lens), B, H, d, n_layers, dtype, align, tail_rows, _p(row_off), _p(o7))
    if rc:
        raise ValueError("upro_layout: invalid argument")
    keys = ["R", "elem_bytes", "row_bytes", "head_stride_bytes", "layer_stride_bytes", "bytes_cache", "bytes_scales"]
    out = {k: int(v) for k, v in zip(keys, o7)}
    out["row_off"] = row_off
    return out


def pack(pool_bits: np.ndarray, slot_ids, seq_lens, dtype: int, align: int = ROW_ALIGN, tail_rows: int = 128):
    """Pool [n_layers,S,H,n_max,d] bf16 bits -> (packed cache bytes, scales or None) (a1)."""
    pool_bits = np.ascontiguousarray(pool_bits, dtype=np.uint16)
    n_layers, S, H, n_max, d = pool_bits.shape
    slot_ids = np.ascontiguousarray(slot_ids, dtype=np.int32)
    seq_lens = np.ascontiguousarray(seq_lens, dtype=np.int32)
    B = int(seq_lens.shape[0])
    lay = layout(seq_lens, H, d, n_layers, dtype, align, tail_rows)
    cache = np.zeros(lay["bytes_cache"], dtype=np.uint8)
    scales = (np.zeros(n_layers * H, dtype=np.float32) if dtype == FP8_E4M3 else
              np.zeros(n_layers * B * H, dtype=np.float32) if dtype == FP8_E4M3_USER else None)
    rc = lib().upro_pack(_p(pool_bits), n_layers, S, H, n_max, d, _p(slot_ids), _p(seq_lens), B, dtype, align,
                         tail_rows, _p(cache), _p(scales))
    if rc:
        raise ValueError("upro_pack: invalid argument")
    return cache, scales


# ---------------------------------------------------------------------------- attention
def attn_block(q, K, V, kself=None, vself=None, scale=None, return_weights: bool = False):
    """One (layer, user, head) block: q [C,d], K/V [L,d], optional kself/vself [C,d] (a2-a7)."""
    q, K, V = _c64(q), _c64(K), _c64(V)
    C, d = q.shape
    L = K.shape[0]
    if scale is None:
        scale = 1.0 / np.sqrt(d)
    ks = _c64(kself) if kself is not None else None
    vs = _c64(vself) if vself is not None else None
    out = np.zeros((C, d), dtype=np.float64)
    w = np.zeros((C, L + 1), dtype=np.float64) if return_weights else None
    lib().upro_attn_block(_p(q), _p(K), _p(V), _p(ks), _p(vs), C, L, d, ctypes.c_double(scale), _p(out), _p(w))
    return (out, w) if return_weights else out


def full_sequence_attention(xq, xk, xv, n: int, k: int, self_flag: bool, scale=None, return_mask: bool = False):
    """Dense masked attention over [history || candidates] as PAPER.md:138 states it."""
    xq, xk, xv = _c64(xq), _c64(xk), _c64(xv)
    T, d = xq.shape
    assert T == n + k
    if scale is None:
        scale = 1.0 / np.sqrt(d)
    out = np.zeros((T, d), dtype=np.float64)
    mask = np.zeros((T, T), dtype=np.uint8) if return_mask else None
    lib().upro_full_sequence_attention(_p(xq), _p(xk), _p(xv), n, k, d, int(bool(self_flag)), ctypes.c_double(scale),
                                       _p(out), _p(mask))
    return (out, mask) if return_mask else out


def attn_partial(q, K, V, j0: int, j1: int, scale=None):
    """Split-K partial state (m, l, O~) of key range [j0, j1) (a8)."""
    q, K, V = _c64(q), _c64(K), _c64(V)
    C, d = q.shape
    if scale is None:
        scale = 1.0 / np.sqrt(d)
    m = np.zeros(C, dtype=np.float64)
    l = np.zeros(C, dtype=np.float64)
    Ot = np.zeros((C, d), dtype=np.float64)
    lib().upro_attn_partial(_p(q), _p(K), _p(V), C, j0, j1, d, ctypes.c_double(scale), _p(m), _p(l), _p(Ot))
    return m, l, Ot


def combine(m, l, Ot):
    """Merge split-K partial states: m, l [P,C], Ot [P,C,d] -> out [C,d] (a8)."""
    m, l, Ot = _c64(m), _c64(l), _c64(Ot)
    P, C, d = Ot.shape
    out = np.zeros((C, d), dtype=np.float64)
    lib().upro_combine(_p(m), _p(l), _p(Ot), P, C, d, _p(out))
    return out


def cross_attn_packed(q, q_dtype: int, k_cache, v_cache, kv_dtype: int, seq_lens, cand_offsets, H: int, d: int,
                      n_layers: int = 1, k_scale=None, v_scale=None, kself=None, vself=None, sm_scale=None,
                      align: int = ROW_ALIGN, users=None):
    """Whole ragged batch in the packed layout (OpenMP over (layer, user, head) blocks).

    q/kself/vself: [n_layers, total_q, H, d] as float32 (F32) or uint16 bf16 bits (BF16).
    k_cache/v_cache: raw packed buffers (float32 / uint16 / uint8 views of [n_layers,H,R,d]).
    Returns out [n_layers, total_q, H, d] float64; rows of users outside ``users`` stay zero.
    """
    seq_lens = np.ascontiguousarray(seq_lens, dtype=np.int32)
    cand_offsets = np.ascontiguousarray(cand_offsets, dtype=np.int32)
    B = int(seq_lens.shape[0])
    total_q = int(cand_offsets[B])
    if sm_scale is None:
        sm_scale = 1.0 / np.sqrt(d)
    qdt = np.float32 if q_dtype == F32 else np.uint16
    kdt = {F32: np.float32, BF16: np.uint16, FP8_E4M3: np.uint8, FP8_E4M3_USER: np.uint8}[kv_dtype]
    q = np.ascontiguousarray(q, dtype=qdt)
    assert q.size == n_layers * total_q * H * d
    k_cache = np.ascontiguousarray(k_cache).view(kdt)
    v_cache = np.ascontiguousarray(v_cache).view(kdt)
    ks = np.ascontiguousarray(kself, dtype=qdt) if kself is not None else None
    vs = np.ascontiguousarray(vself, dtype=qdt) if vself is not None else None
    ksc = np.ascontiguousarray(k_scale, dtype=np.float32) if k_scale is not None else None
    vsc = np.ascontiguousarray(v_scale, dtype=np.float32) if v_scale is not None else None
    lo, hi = (0, B) if users is None else users
    out = np.zeros((n_layers, total_q, H, d), dtype=np.float64)
    rc = lib().upro_cross_attn_packed(_p(q), q_dtype, _p(k_cache), _p(v_cache), kv_dtype, _p(ksc), _p(vsc), _p(ks),
                                      _p(vs), _p(seq_lens), _p(cand_offsets), B, H, d, n_layers, align,
                                      ctypes.c_double(sm_scale), lo, hi, _p(out))
    if rc:
        raise ValueError("upro_cross_attn_packed: invalid argument")
    return out


def cross_attn_pool(q, q_dtype: int, k_pool_bits, v_pool_bits, slot_ids, seq_lens, cand_offsets, H_q: int,
                    kself=None, vself=None, sm_scale=None, users=None):
    """Whole ragged batch read straight from the pool [n_layers,S,H_kv,n_max,d] (bf16 bits), no pack
    (zero-copy addressing); H_q may be a multiple of H_kv (grouped queries: head hq -> KV head hq // G).
    Returns out [n_layers, total_q, H_q, d] float64; rows of users outside ``users`` stay zero."""
    k_pool_bits = np.ascontiguousarray(k_pool_bits, dtype=np.uint16)
    v_pool_bits = np.ascontiguousarray(v_pool_bits, dtype=np.uint16)
    n_layers, S, H_kv, n_max, d = k_pool_bits.shape
    assert v_pool_bits.shape == k_pool_bits.shape
    slot_ids = np.ascontiguousarray(slot_ids, dtype=np.int32)
    seq_lens = np.ascontiguousarray(seq_lens, dtype=np.int32)
    cand_offsets = np.ascontiguousarray(cand_offsets, dtype=np.int32)
    B = int(seq_lens.shape[0])
    total_q = int(cand_offsets[B])
    if sm_scale is None:
        sm_scale = 1.0 / np.sqrt(d)
    qdt = np.float32 if q_dtype == F32 else np.uint16
    q = np.ascontiguousarray(q, dtype=qdt)
    assert q.size == n_layers * total_q * H_q * d
    ks = np.ascontiguousarray(kself, dtype=qdt) if kself is not None else None
    vs = np.ascontiguousarray(vself, dtype=qdt) if vself is not None else None
    lo, hi = (0, B) if users is None else users
    out = np.zeros((n_layers, total_q, H_q, d), dtype=np.float64)
    rc = lib().upro_cross_attn_pool(_p(q), q_dtype, _p(k_pool_bits), _p(v_pool_bits), n_layers, S, H_kv, n_max, d,
                                    H_q, _p(slot_ids), _p(seq_lens), _p(cand_offsets), B, _p(ks), _p(vs),
                                    ctypes.c_double(sm_scale), lo, hi, _p(out))
    if rc:
        raise ValueError("upro_cross_attn_pool: invalid argument")
    return out


# ---------------------------------------------------------------------------- decode-layer tail, consumer
ACT_NONE, ACT_SILU, ACT_RELU = 0, 1, 2


def linear(x, w, b=None, act: int = ACT_NONE):
    """y = act(x W^T + b) in fp64; x [M,K], w [N,K] (nn.Linear convention), b [N] or None."""
    x, w = _c64(x), _c64(w)
    M, K = x.shape
    N = w.shape[0]
    assert w.shape[1] == K
    bb = _c64(b) if b is not None else None
    y = np.zeros((M, N), dtype=np.float64)
    lib().upro_linear(_p(x), _p(w), _p(bb), ctypes.c_int64(M), N, K, act, _p(y))
    return y


def action_utility(z, w1, b1, w2, b2, wc, act: int = ACT_SILU):
    """Per-action MLP heads -> probabilities -> weighted utility.
    z [M,D]; w1 [C,Dh,D]; b1 [C,Dh]; w2 [C,Dh]; b2 [C]; wc [C].  Returns (probs [M,C], util [M])."""
    z, w1, b1, w2, b2, wc = (_c64(a) for a in (z, w1, b1, w2, b2, wc))
    M, D = z.shape
    C, Dh, _ = w1.shape
    probs = np.zeros((M, C), dtype=np.float64)
    util = np.zeros(M, dtype=np.float64)
    lib().upro_action_utility(_p(z), _p(w1), _p(b1), _p(w2), _p(b2), _p(wc), ctypes.c_int64(M), D, C, Dh, act,
                              _p(probs), _p(util))
    return probs, util


def topk_per_user(util, cand_offsets, K: int):
    """Top-K candidates per user by utility (fp32 compare), ties by ascending index.
    Returns (idx [B,K] int32 global candidate indices, -1 padded; cnt [B] int32)."""
    util = np.ascontiguousarray(util, dtype=np.float32)
    cand_offsets = np.ascontiguousarray(cand_offsets, dtype=np.int32)
    B = int(cand_offsets.shape[0]) - 1
    idx = np.zeros((B, K), dtype=np.int32)
    cnt = np.zeros(B, dtype=np.int32)
    lib().upro_topk_per_user(_p(util), _p(cand_offsets), B, K, _p(idx), _p(cnt))
    return idx, cnt


def layernorm(x, gamma, beta, eps: float = 1e-5):
    """y = (x - mean) / sqrt(var + eps) * gamma + beta over the last axis, fp64; x [M,D]."""
    x, gamma, beta = _c64(x), _c64(gamma), _c64(beta)
    M, D = x.shape
    y = np.zeros((M, D), dtype=np.float64)
    lib().upro_layernorm(_p(x), _p(gamma), _p(beta), ctypes.c_int64(M), D, ctypes.c_double(eps), _p(y))
    return y


def linear_fp8(x, x_scale: float, w8, w_scale: float, b=None, act: int = ACT_NONE):
    """FP8 E4M3 linear layer with fused per-tensor scaling: x [M,K] float32 values, w8 [N,K] E4M3 bytes."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    w8 = np.ascontiguousarray(w8, dtype=np.uint8)
    M, K = x.shape
    N = w8.shape[0]
    bb = _c64(b) if b is not None else None
    y = np.zeros((M, N), dtype=np.float64)
    lib().upro_linear_fp8(_p(x), ctypes.c_float(x_scale), _p(w8), ctypes.c_float(w_scale), _p(bb), ctypes.c_int64(M), N, K,
                          act, _p(y))
    return y


def linear_fp8q(x8, x_scale: float, w8, w_scale: float, b=None, act: int = ACT_NONE):
    """FP8 E4M3 linear layer whose activations arrive as E4M3 bytes: x8 [M,K], w8 [N,K] E4M3 bytes."""
    x8 = np.ascontiguousarray(x8, dtype=np.uint8)
    w8 = np.ascontiguousarray(w8, dtype=np.uint8)
    M, K = x8.shape
    N = w8.shape[0]
    bb = _c64(b) if b is not None else None
    y = np.zeros((M, N), dtype=np.float64)
    lib().upro_linear_fp8q(_p(x8), ctypes.c_float(x_scale), _p(w8), ctypes.c_float(w_scale), _p(bb), ctypes.c_int64(M), N,
                           K, act, _p(y))
    return y
