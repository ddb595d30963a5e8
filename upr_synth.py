"""Seeded synthetic inputs for the ranking cross-attention path (serves BOTH the oracle
tests and the CUDA path; holds none of the method's arithmetic).

The paper's workloads are Pinterest-internal (B=8, n=992, k=656, 12 layers;
PAPER.md:309: histories of 256..2048 tokens; up to ~3000 candidates), so
the BASELINE.json configs stand in for them: ragged histories, hundreds to a thousand
candidates per user, multi-layer caches, unit-variance q/K/V.

Generator: a counter-based hash, splitmix64(key(seed, tag) +
(i+1)*gamma), evaluated with wrapping int64 arithmetic so that the same element comes out
bit-identically on CPU and on CUDA and independently of generation order.  Normal draws
take 16 hash bits as an index into a 65536-entry table of N(0,1) quantiles
ndtri((i+0.5)/65536) rounded once to bf16 (the table is always computed on the CPU).
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np
import torch

_M64 = (1 << 64) - 1
_GAMMA = 0x9E3779B97F4A7C15
_C1 = 0xBF58476D1CE4E5B9
_C2 = 0x94D049BB133111EB


def _s64(x: int) -> int:
    """Two's-complement view of a uint64 as a Python int that fits torch.int64."""
    x &= _M64
    return x - (1 << 64) if x >= (1 << 63) else x


def splitmix64(x: int) -> int:
    """Reference scalar splitmix64 finaliser on Python ints (uint64 semantics)."""
    z = (x + _GAMMA) & _M64
    z = ((z ^ (z >> 30)) * _C1) & _M64
    z = ((z ^ (z >> 27)) * _C2) & _M64
    return z ^ (z >> 31)


def stream_key(seed: int, tag: str) -> int:
    k = splitmix64(seed & _M64)
    for ch in tag.encode():
        k = splitmix64(k ^ ch)
    return k


def _lsr(z: torch.Tensor, s: int) -> torch.Tensor:
    return torch.bitwise_and(torch.bitwise_right_shift(z, s), (1 << (64 - s)) - 1)


def hash_u64(key: int, start: int, n: int, device) -> torch.Tensor:
    """Element i (start <= i < start+n) of stream ``key`` as int64 holding uint64 bits."""
    i = torch.arange(start + 1, start + n + 1, dtype=torch.int64, device=device)
    z = i * _s64(_GAMMA) + _s64(key)  # state = key + (i+1)*gamma  (wraps)
    z = z + _s64(_GAMMA)
    z = (z ^ _lsr(z, 30)) * _s64(_C1)
    z = (z ^ _lsr(z, 27)) * _s64(_C2)
    return z ^ _lsr(z, 31)


def hash_u64_scalar(key: int, i: int) -> int:
    return splitmix64((key + (i + 1) * _GAMMA) & _M64)


_TABLE: Optional[torch.Tensor] = None


def normal_table_bf16() -> torch.Tensor:
    """65536 N(0,1) quantiles rounded to bf16 (CPU tensor, computed once in fp64)."""
    global _TABLE
    if _TABLE is None:
        p = (torch.arange(65536, dtype=torch.float64) + 0.5) / 65536.0
        _TABLE = torch.special.ndtri(p).to(torch.float32).to(torch.bfloat16)
    return _TABLE


def normal_bf16(seed: int, tag: str, shape, device="cpu", chunk: int = 1 << 25) -> torch.Tensor:
    """N(0,1) draws stored as bf16, bit-identical on every device."""
    n = int(np.prod(shape))
    key = stream_key(seed, tag)
    table = normal_table_bf16().to(device)
    out = torch.empty(n, dtype=torch.bfloat16, device=device)
    for s in range(0, n, chunk):
        m = min(chunk, n - s)
        idx = torch.bitwise_and(_lsr(hash_u64(key, s, m, device), 40), 0xFFFF)
        out[s:s + m] = table[idx]
    return out.view(*shape)


def normal_f32(seed: int, tag: str, shape) -> torch.Tensor:
    """fp32 N(0,1) draws for the fp32 toy config (CPU; 32 hash bits -> ndtri in fp64)."""
    n = int(np.prod(shape))
    key = stream_key(seed, tag)
    h = _lsr(hash_u64(key, 0, n, "cpu"), 32).to(torch.float64)
    p = (h + 0.5) / 4294967296.0
    return torch.special.ndtri(p).to(torch.float32).view(*shape)


def uniform_ints(seed: int, tag: str, n: int, lo: int, hi: int) -> np.ndarray:
    """n integers uniform on [lo, hi] (inclusive)."""
    key = stream_key(seed, tag)
    span = hi - lo + 1
    return np.array([lo + hash_u64_scalar(key, i) % span for i in range(n)], dtype=np.int32)


def log_uniform_ints(seed: int, tag: str, n: int, lo: int, hi: int) -> np.ndarray:
    """floor(lo * (hi/lo)**u), u uniform on [0,1), clipped to [lo, hi]."""
    key = stream_key(seed, tag)
    out = np.empty(n, dtype=np.int32)
    ratio = math.log2(hi / lo)
    for i in range(n):
        u = (hash_u64_scalar(key, i) >> 11) / float(1 << 53)
        out[i] = min(hi, max(lo, int(math.floor(lo * 2.0 ** (ratio * u)))))
    return out


def permutation(seed: int, tag: str, n: int) -> np.ndarray:
    key = stream_key(seed, tag)
    keys = np.array([hash_u64_scalar(key, i) for i in range(n)], dtype=np.uint64)
    return np.argsort(keys, kind="stable").astype(np.int32)


# ------------------------------------------------------------------------------ workloads
@dataclasses.dataclass
class Workload:
    name: str
    seed: int
    B: int
    H: int
    d: int
    n_layers: int
    seq_lens: np.ndarray       # [B] int32  history length L_b  (paper: n)
    cand_offsets: np.ndarray   # [B+1] int32 exclusive prefix of candidate counts C_b (paper: k)
    kv_dtype: str              # "f32" | "bf16" | "fp8"
    q_dtype: str               # "f32" | "bf16"
    self_term: bool
    n_max: int                 # pool slot length (paper's n in [L,S,H,n,D])
    cfg: object = None         # BASELINE.json config id this workload was built from

    @property
    def total_q(self) -> int:
        return int(self.cand_offsets[-1])

    @property
    def cand_counts(self) -> np.ndarray:
        return np.diff(self.cand_offsets).astype(np.int64)

    @property
    def pairs(self) -> int:
        """(query, key) pairs over all layers and heads (self pairs excluded)."""
        return int((self.cand_counts * self.seq_lens.astype(np.int64)).sum()) * self.H * self.n_layers

    @property
    def flops(self) -> int:
        f = 4 * self.d * self.pairs
        if self.self_term:
            f += 4 * self.d * self.total_q * self.H * self.n_layers
        return f

    def kv_elem_bytes(self) -> int:
        return {"f32": 4, "bf16": 2, "fp8": 1, "fp8_user": 1}[self.kv_dtype]

    @property
    def kv_bytes(self) -> int:
        """Algorithmic K+V cache bytes: every valid row once per (layer, head)."""
        return int(self.seq_lens.astype(np.int64).sum()) * self.H * self.d * self.n_layers * 2 * self.kv_elem_bytes()


def _offsets(counts) -> np.ndarray:
    return np.concatenate([[0], np.cumsum(np.asarray(counts, dtype=np.int64))]).astype(np.int32)


def workload(cfg: int | str, users: Optional[int] = None) -> Workload:
    """The five BASELINE.json configs (1..5) and the supplementary low-C shape "S1".
    ``users`` overrides B (same per-user distributions) for reduced-size parity cases."""
    w = _workload(cfg, users)
    w.cfg = cfg
    return w


def _workload(cfg, users):
    if cfg == 1:
        B = users or 1
        return Workload("cfg1_fp32_toy", 1001, B, 4, 64, 1, np.full(B, 256, np.int32), _offsets([16] * B),
                        "f32", "f32", False, 256)
    if cfg == 2:
        B = users or 64
        L = uniform_ints(1002, "seq_lens", B, 128, 1024)
        return Workload("cfg2_bf16_B64", 1002, B, 8, 64, 1, L, _offsets([256] * B), "bf16", "bf16", False, 1024)
    if cfg == 3:
        B = users or 256
        L = uniform_ints(1003, "seq_lens", B, 512, 2048)
        return Workload("cfg3_bf16_B256_4layer", 1003, B, 8, 128, 4, L, _offsets([512] * B), "bf16", "bf16",
                        False, 2048)
    if cfg == 4:
        B = users or 128
        return Workload("cfg4_fp8_B128_2layer", 1004, B, 16, 64, 2, np.full(B, 4096, np.int32),
                        _offsets([1000] * B), "fp8", "bf16", False, 4096)
    if cfg == 5:
        B = users or 512
        L = log_uniform_ints(1005, "seq_lens", B, 64, 8192)
        C = uniform_ints(1005, "cand_counts", B, 50, 1000)
        return Workload("cfg5_serving_mix", 1005, B, 8, 128, 1, L, _offsets(C), "bf16", "bf16", True, 8192)
    if cfg == "S1":
        B = users or 512
        return Workload("S1_lowC_membound", 1006, B, 8, 128, 1, np.full(B, 4096, np.int32), _offsets([32] * B),
                        "bf16", "bf16", False, 4096)
    raise ValueError(f"unknown config {cfg!r}")


def slot_ids(w: Workload) -> np.ndarray:
    """S = B pool slots, users mapped through a seeded permutation (round-robin reuse)."""
    return permutation(w.seed, "slot_ids", w.B)


def gen_queries(w: Workload, tag: str = "q", device="cpu", scale: float = 1.0) -> torch.Tensor:
    """[n_layers, total_q, H, d] candidate-side tensor (q, k_self or v_self)."""
    shape = (w.n_layers, w.total_q, w.H, w.d)
    if w.q_dtype == "f32":
        t = normal_f32(w.seed, tag, shape).to(device)
    else:
        t = normal_bf16(w.seed, tag, shape, device)
    if scale != 1.0:
        t = (t.float() * scale).to(t.dtype)
    return t


def gen_pool(w: Workload, tag: str, device="cpu") -> torch.Tensor:
    """The paper's KV pool [n_layers, S=B, H, n_max, d] in bf16."""
    return normal_bf16(w.seed, tag, (w.n_layers, w.B, w.H, w.n_max, w.d), device)


def custom_workload(name: str, seed: int, seq_lens, cand_counts, H: int, d: int, n_layers: int = 1,
                    kv_dtype: str = "bf16", q_dtype: str = "bf16", self_term: bool = False,
                    n_max: Optional[int] = None) -> Workload:
    """Arbitrary ragged shape for edge-case parity tests."""
    L = np.asarray(seq_lens, dtype=np.int32)
    n_max = n_max or max(1, int(L.max()) if L.size else 1)
    return Workload(name, seed, int(L.shape[0]), H, d, n_layers, L, _offsets(cand_counts), kv_dtype, q_dtype,
                    self_term, n_max)
