"""Shared helpers for the GPU parity tests: build seeded inputs, run the CUDA path through the
C-ABI binding, run the oracle on the SAME stored input values (never on CUDA outputs)."""
from __future__ import annotations

import numpy as np
import torch

import oracle
import upr_synth as S

ORACLE_DT = {"f32": oracle.F32, "bf16": oracle.BF16, "fp8": oracle.FP8_E4M3, "fp8_user": oracle.FP8_E4M3_USER}


def bits(t: torch.Tensor) -> np.ndarray:
    """bf16 tensor -> uint16 bit patterns on the host; fp32 tensor -> float32 array."""
    t = t.detach().cpu().contiguous()
    if t.dtype == torch.bfloat16:
        return t.view(torch.int16).numpy().view(np.uint16)
    return t.numpy()


def to_f64(t: torch.Tensor) -> np.ndarray:
    return t.detach().cpu().to(torch.float64).numpy()


class Inputs:
    def __init__(self, w: S.Workload, device, q_scale: float = 1.0, H_kv=None):
        """w.H is the number of QUERY heads; H_kv (default w.H) the number of KV heads of the pool
        (grouped queries: query head hq reads KV head hq // (w.H // H_kv), "KV heads")."""
        self.w = w
        self.device = device
        self.H_kv = H_kv or w.H
        self.G = w.H // self.H_kv
        assert self.G * self.H_kv == w.H
        self.q = S.gen_queries(w, "q", device, q_scale)
        self.k_self = S.gen_queries(w, "k_self", device) if w.self_term else None
        self.v_self = S.gen_queries(w, "v_self", device) if w.self_term else None
        pool_shape = (w.n_layers, w.B, self.H_kv, w.n_max, w.d)
        self.k_pool = S.normal_bf16(w.seed, "k_pool", pool_shape, device)   # == S.gen_pool when H_kv == w.H
        self.v_pool = S.normal_bf16(w.seed, "v_pool", pool_shape, device)
        self.slot_ids_host = S.slot_ids(w)
        self.slot_ids = torch.as_tensor(self.slot_ids_host, device=device)

    def block_kv_f64(self, l: int, b: int, h: int):
        """History K/V rows of one (layer, user, head) block, straight from the generated pool
        (bf16 values widened exactly) -- for bf16/f32 caches this IS what the cache stores."""
        Lb = int(self.w.seq_lens[b])
        s = int(self.slot_ids_host[b])
        hk = h // self.G
        return to_f64(self.k_pool[l, s, hk, :Lb]), to_f64(self.v_pool[l, s, hk, :Lb])

    def oracle_fp8_cache(self):
        """(k_bytes, k_scale, v_bytes, v_scale, row_off, R): the ORACLE's E4M3 pack of the whole pools
        (small workloads only: the oracle's nearest-code search costs ~0.1 us per element)."""
        if not hasattr(self, "_fp8"):
            kc, ks = oracle.pack(bits(self.k_pool), self.slot_ids_host, self.w.seq_lens, oracle.FP8_E4M3)
            vc, vs = oracle.pack(bits(self.v_pool), self.slot_ids_host, self.w.seq_lens, oracle.FP8_E4M3)
            lay = oracle.layout(self.w.seq_lens, self.w.H, self.w.d, self.w.n_layers, oracle.FP8_E4M3)
            self._fp8 = (kc, ks, vc, vs, lay["row_off"], lay["R"])
        return self._fp8

    def _oracle_fp8_head(self, l: int, h: int):
        """The oracle's E4M3 pack of ONE (layer, head) slice of the pools, all users: the scale is
        per (layer, head) over every user's valid rows, so this slice is self-contained."""
        cache = self.__dict__.setdefault("_fp8_head", {})
        if (l, h) not in cache:
            kp = bits(self.k_pool[l:l + 1, :, h:h + 1])
            vp = bits(self.v_pool[l:l + 1, :, h:h + 1])
            kc, ks = oracle.pack(kp, self.slot_ids_host, self.w.seq_lens, oracle.FP8_E4M3)
            vc, vs = oracle.pack(vp, self.slot_ids_host, self.w.seq_lens, oracle.FP8_E4M3)
            lay = oracle.layout(self.w.seq_lens, 1, self.w.d, 1, oracle.FP8_E4M3)
            cache.clear()                                  # keep one slice at a time
            cache[(l, h)] = (kc, float(ks[0]), vc, float(vs[0]), lay["row_off"])
        return cache[(l, h)]

    def block_kv_dequant_f64(self, l: int, b: int, h: int):
        """History K/V of one block as the FP8 cache stores them: decode(byte) * scale, exact in fp64."""
        kc, ks, vc, vs, row_off = self._oracle_fp8_head(l, h)
        d, Lb = self.w.d, int(self.w.seq_lens[b])
        r0 = int(row_off[b]) * d
        K = oracle.e4m3_decode(kc[r0:r0 + Lb * d]).reshape(Lb, d) * ks
        V = oracle.e4m3_decode(vc[r0:r0 + Lb * d]).reshape(Lb, d) * vs
        return K, V

    def block_q_f64(self, l: int, b: int, h: int):
        co = self.w.cand_offsets
        sl = slice(int(co[b]), int(co[b + 1]))
        q = to_f64(self.q[l, sl, h])
        if self.k_self is None:
            return q, None, None
        return q, to_f64(self.k_self[l, sl, h]), to_f64(self.v_self[l, sl, h])


def oracle_block(inp: Inputs, l: int, b: int, h: int, sm_scale=None, dequant: bool = False) -> np.ndarray:
    K, V = inp.block_kv_dequant_f64(l, b, h) if dequant else inp.block_kv_f64(l, b, h)
    q, ks, vs = inp.block_q_f64(l, b, h)
    return oracle.attn_block(q, K, V, ks, vs, scale=sm_scale)


def oracle_all(inp: Inputs, sm_scale=None, dequant: bool = False) -> np.ndarray:
    w = inp.w
    out = np.zeros((w.n_layers, w.total_q, w.H, w.d))
    co = w.cand_offsets
    for l in range(w.n_layers):
        for h in range(w.H):
            for b in range(w.B):
                if co[b + 1] == co[b]:
                    continue
                out[l, co[b]:co[b + 1], h] = oracle_block(inp, l, b, h, sm_scale, dequant)
    return out


def error_stats(got: np.ndarray, want: np.ndarray):
    diff = np.abs(got.astype(np.float64) - want)
    rms = float(np.sqrt(np.mean(want ** 2))) or 1.0
    return float(diff.max()) if diff.size else 0.0, float(np.sqrt(np.mean(diff ** 2)) / rms) if diff.size else 0.0
