#!/usr/bin/env python
"""bench.py -- ranking cross-attention candidates/s on one node (driver contract).

One "step" is one pass of the whole hot path over one batch of
synthetic input: layout (host integers) -> pack the users' pool slots into the decode cache
 -> cross-attention of every candidate over its user's cached history for all
layers [-> split-K combine when the split policy engages].

    python bench.py --gpus N --steps K --warmup W [--config 3] [--impl reference]

N = 1: BASELINE.json config 3 (largest bf16 config, the one the 60%-of-roofline target names).
N > 1 (torchrun): users are independent, so every rank runs its own batch of
the same config with a rank-specific seed -- weak scaling, no data-path collective.
Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import upr_synth as S  # noqa: E402

METRIC = "ranking cross-attn candidates/sec/GPU; TFLOP/s as fraction of roofline"


# ----------------------------------------------------------------------------- helpers
def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return {"hbm_gbs": p["hbm_gbs"], "bf16_tflops": p["bf16_tflops"],
                "bf16_tflops_sustained": p.get("bf16_tflops_sustained", p["bf16_tflops"]), "source": "measured"}
    # fallback stated in B200_PROFILING.md
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "source": "fallback"}


class ClockSampler:
    """SM clock, power and throttle reasons polled through NVML every ~5 ms DURING the timed
    region (nvidia-smi -lms is too coarse for a sub-second region)."""

    def __init__(self, index: int):
        self.index = index
        self.samples = []
        self.stop_flag = threading.Event()
        self.thread = None
        self.nv = None
        self.err = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(self._physical_index(index))
        except Exception as e:  # noqa: BLE001 -- no NVML: report it, never fail the bench
            self.nv, self.err = None, repr(e)

    @staticmethod
    def _physical_index(index: int) -> int:
        vis = os.environ.get("CUDA_VISIBLE_DEVICES")
        if vis:
            ids = [x for x in vis.split(",") if x.strip()]
            if index < len(ids) and ids[index].strip().isdigit():
                return int(ids[index])
        return index

    def _poll(self):
        nv = self.nv
        while not self.stop_flag.is_set():
            try:
                sm = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
                pw = nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0
                rs = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                self.samples.append((sm, pw, rs))
            except Exception as e:  # noqa: BLE001
                self.err = repr(e)
                break
            time.sleep(0.005)

    def start(self):
        if self.nv is not None:
            self.thread = threading.Thread(target=self._poll, daemon=True)
            self.thread.start()

    def stop(self):
        if self.nv is None or self.thread is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml unavailable: %s" % self.err]}
        self.stop_flag.set()
        self.thread.join(timeout=2)
        nv = self.nv
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples: %s" % self.err]}
        try:
            mx = float(nv.nvmlDeviceGetMaxClockInfo(self.h, nv.NVML_CLOCK_SM))
        except Exception:  # noqa: BLE001
            mx = None
        bits = {"hw_slowdown": nv.nvmlClocksEventReasonHwSlowdown,
                "hw_thermal_slowdown": nv.nvmlClocksEventReasonHwThermalSlowdown,
                "sw_thermal_slowdown": nv.nvmlClocksEventReasonSwThermalSlowdown,
                "sw_power_cap": nv.nvmlClocksEventReasonSwPowerCap}
        reasons = sorted(k for k, b in bits.items() if any(r & b for _, _, r in self.samples))
        return {"sm_mhz": float(np.median([s[0] for s in self.samples])), "sm_max_mhz": mx,
                "sm_min_mhz": float(min(s[0] for s in self.samples)),
                "power_w_max": float(max(s[1] for s in self.samples)), "samples": len(self.samples),
                "reasons": reasons, "how": "NVML polled every 5 ms inside the timed region"}


def aggregate_over_ranks(local_ms: float, local_units: int, dist=None):
    """Whole-job numbers from per-rank ones: time = max over ranks, units = sum over ranks.
    Works on any backend (nccl on GPU, gloo in the CPU test)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return local_ms, local_units
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([local_ms], dtype=torch.float64, device=dev)
    u = torch.tensor([local_units], dtype=torch.int64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), int(u.item())


def rank_workload(cfg, rank: int) -> S.Workload:
    """Rank r's batch: same config, rank-specific seed (users are independent units)."""
    w = S.workload(cfg)
    if rank:
        w.seed = w.seed + 7919 * rank
    return w


# ----------------------------------------------------------------------------- oracle legs
def oracle_step(w: S.Workload, users: int):
    """One oracle pass (pack + attention, all layers/heads) over the first `users` users.
    Returns (seconds, candidates processed)."""
    import oracle
    sub = S.workload(w.cfg, users=users)
    dt = {"f32": oracle.F32, "bf16": oracle.BF16, "fp8": oracle.FP8_E4M3}[sub.kv_dtype]
    qdt = oracle.F32 if sub.q_dtype == "f32" else oracle.BF16

    def b(t):
        t = t.contiguous()
        return t.view(torch.int16).numpy().view(np.uint16) if t.dtype == torch.bfloat16 else t.numpy()
    q = b(S.gen_queries(sub, "q"))
    ks = b(S.gen_queries(sub, "k_self")) if sub.self_term else None
    vs = b(S.gen_queries(sub, "v_self")) if sub.self_term else None
    kp, vp = b(S.gen_pool(sub, "k_pool")), b(S.gen_pool(sub, "v_pool"))
    slots = S.slot_ids(sub)
    t0 = time.perf_counter()
    kc, ksc = oracle.pack(kp, slots, sub.seq_lens, dt)
    vc, vsc = oracle.pack(vp, slots, sub.seq_lens, dt)
    oracle.cross_attn_packed(q, qdt, kc, vc, dt, sub.seq_lens, sub.cand_offsets, sub.H, sub.d, sub.n_layers,
                             ksc, vsc, ks, vs)
    return time.perf_counter() - t0, sub.total_q


def oracle_sample_users(w: S.Workload, budget_s: float) -> int:
    t1, _ = oracle_step(w, 1)
    return int(max(1, min(w.B, budget_s / max(t1, 1e-3))))


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    w = S.workload(args.config)
    users = oracle_sample_users(w, 6.0)
    for _ in range(args.warmup):
        oracle_step(w, users)
    ts, cands = [], 0
    for _ in range(args.steps):
        t, cands = oracle_step(w, users)
        ts.append(t)
    ms = 1e3 * float(np.mean(ts))
    val = cands / (ms * 1e-3)
    sample = f"first {users} of {w.B} users of {w.name}, all layers and heads, pack + attention"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "candidates/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "sample": sample},
            "cpu_baseline": {"value": val, "unit": "candidates/s", "cores": oracle.num_threads(), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": val, "unit": "candidates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


# ----------------------------------------------------------------------------- ranking tail
def ranking_tail(P, w, attn, q, k_self, v_self, q_host, stream, dev, ev, n_heads=4, d_head_hidden=128, top_k=100,
                 iters=5):
    """Synthetic-weight tail of the ranking pass on the last layer's attention output.
    Returns per-kernel times, GEMM TFLOP/s and an end-to-end figure where only the top-K indices return to the host."""
    import math
    D = w.H * w.d
    M = w.total_q

    def wgt(tag, n, k):
        return (S.normal_bf16(w.seed, tag, (n, k), dev).float() / math.sqrt(k)).to(torch.bfloat16)
    w_o, w_1 = wgt("w_o", D, D), wgt("w_head1", n_heads * d_head_hidden, D)
    b_1 = torch.zeros(n_heads * d_head_hidden, dtype=torch.float32, device=dev)
    w_2 = S.normal_bf16(w.seed, "w_head2", (n_heads, d_head_hidden), dev).float() / math.sqrt(d_head_hidden)
    b_2 = torch.zeros(n_heads, dtype=torch.float32, device=dev)
    w_c = torch.ones(n_heads, dtype=torch.float32, device=dev)
    z = torch.empty((M, D), dtype=torch.bfloat16, device=dev)
    hid = torch.empty((M, n_heads * d_head_hidden), dtype=torch.bfloat16, device=dev)
    util = torch.empty(M, dtype=torch.float32, device=dev)
    idx = torch.empty((w.B, top_k), dtype=torch.int32, device=dev)
    cnt = torch.empty(w.B, dtype=torch.int32, device=dev)
    idx_host = torch.empty((w.B, top_k), dtype=torch.int32).pin_memory()
    max_c = int(w.cand_counts.max())
    marks = [ev() for _ in range(5)]

    def tail_once(out_last, record=False):
        x = out_last.view(M, D)
        if record:
            marks[0].record(stream)
        P.upr_linear_fwd(x, w_o, None, z, P.UPR_ACT_NONE, stream)                 # out-projection
        if record:
            marks[1].record(stream)
        P.upr_linear_fwd(z, w_1, b_1, hid, P.UPR_ACT_SILU, stream)                # heads, first layers
        if record:
            marks[2].record(stream)
        P.upr_action_utility(hid, w_2, b_2, w_c, None, util, stream)              # logits -> probabilities -> utility
        if record:
            marks[3].record(stream)
        P.upr_topk_per_user(util, attn.cand_offsets, top_k, max_c, idx, cnt, stream)
        if record:
            marks[4].record(stream)
    out = attn(q, k_self, v_self, stream=stream)
    for _ in range(2):
        tail_once(out[-1])
    torch.cuda.synchronize()
    ts = np.zeros(4)
    for _ in range(iters):
        tail_once(out[-1], record=True)
        torch.cuda.synchronize()
        ts += np.array([marks[i].elapsed_time(marks[i + 1]) for i in range(4)])
    ts /= iters
    # end to end, ranked: queries up, attention + tail on the device, K indices per user back
    q_dev = torch.empty_like(q)
    e0, e1 = ev(), ev()
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(iters):
        q_dev.copy_(q_host, non_blocking=True)
        o = attn(q_dev, k_self, v_self, stream=stream)
        tail_once(o[-1])
        idx_host.copy_(idx, non_blocking=True)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / iters
    assert int(idx_host.max()) < M and int(cnt.min()) >= 0
    fl_o, fl_h = 2.0 * M * D * D, 2.0 * M * D * n_heads * d_head_hidden
    return {"shapes": {"M": M, "D_model": D, "action_heads": n_heads, "head_hidden": d_head_hidden, "top_k": top_k},
            "out_proj_ms": float(ts[0]), "out_proj_tflops": fl_o / (ts[0] * 1e-3) / 1e12,
            "heads_gemm_ms": float(ts[1]), "heads_gemm_tflops": fl_h / (ts[1] * 1e-3) / 1e12,
            "utility_ms": float(ts[2]), "utility_gbs": (hid.numel() * 2 + M * 4) / (ts[2] * 1e-3) / 1e9,
            "topk_ms": float(ts[3]),
            "e2e_ranked": {"value": M / (ms * 1e-3), "unit": "candidates/s", "ms_per_step": ms,
                           "h2d_bytes_per_step": q_host.numel() * q_host.element_size(),
                           "d2h_bytes_per_step": idx_host.numel() * 4,
                           "what": "q up, all layers' attention + out-projection + action heads + utility + top-K on the "
                                   "device, K indices per user back"}}


def decode_layer_leg(P, pl, w, k_pool, v_pool, slots, stream, dev, ev, hidden_mult=4, iters=5):
    """One whole pre-LN decode layer over all candidates of the batch (layer 0's K/V, read in place; synthetic
    weights; self key/value from the layer's own projections): LN, Q / self-K,V projections, cross-attention,
    out-projection + residual, LN, MLP + residual -- pipeline.RankingDecodeLayer, C-ABI calls only."""
    import math
    D, M = w.H * w.d, w.total_q
    hidden = hidden_mult * D

    def wgt(tag, n, k):
        return (S.normal_bf16(w.seed, tag, (n, k), dev).float() / math.sqrt(k)).to(torch.bfloat16)
    ones, zeros = torch.ones(D, device=dev), torch.zeros(D, device=dev)
    prm = {"ln1_g": ones, "ln1_b": zeros, "ln2_g": ones, "ln2_b": zeros, "wq": wgt("dl_wq", D, D), "wk": wgt("dl_wk", D, D),
           "wv": wgt("dl_wv", D, D), "wo": wgt("dl_wo", D, D), "w1": wgt("dl_w1", hidden, D), "w2": wgt("dl_w2", D, hidden),
           "b1": torch.zeros(hidden, device=dev), "b2": zeros}
    view = pl.PoolView.of(k_pool[:1], v_pool[:1], slots, w.seq_lens)
    attn1 = pl.CrossAttention(view, w.cand_offsets, P.UPR_BF16, num_splits=0)
    layer = pl.RankingDecodeLayer(attn1, D, hidden, prm)
    x = S.normal_bf16(w.seed, "dl_x", (M, D), dev)
    for _ in range(2):
        layer(x, stream=stream)
    torch.cuda.synchronize()
    e0, e1 = ev(), ev()
    e0.record(stream)
    for _ in range(iters):
        layer(x, stream=stream)
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / iters
    # the MLP's up-projection alone, bf16 operands vs FP8 E4M3 operands with fused scaling
    def time_it(fn):
        fn(); fn()
        torch.cuda.synchronize()
        a0, a1 = ev(), ev()
        a0.record(stream)
        for _ in range(iters):
            fn()
        a1.record(stream)
        torch.cuda.synchronize()
        return a0.elapsed_time(a1) / iters
    w1f = prm["w1"].float()
    w_scale = float(w1f.abs().max().item()) / 448.0
    w1_8 = (w1f / w_scale).to(torch.float8_e4m3fn).view(torch.uint8)
    up_bf16 = time_it(lambda: P.upr_linear_fwd(layer.h2, prm["w1"], prm["b1"], layer.u, P.UPR_ACT_SILU, stream))
    up_fp8 = time_it(lambda: P.upr_linear_fp8_fwd(layer.h2, 6.0 / 448.0, w1_8, w_scale, prm["b1"], None, layer.u,
                                                  P.UPR_ACT_SILU, stream))
    # the whole MLP as an FP8 chain: up-projection leaves E4M3 bytes, the down-projection reads them through TMA
    w2f = prm["w2"].float()
    w2_scale = float(w2f.abs().max().item()) / 448.0
    w2_8 = (w2f / w2_scale).to(torch.float8_e4m3fn).view(torch.uint8)
    u8 = torch.empty((M, hidden), dtype=torch.uint8, device=dev)
    y8 = torch.empty((M, D), dtype=torch.bfloat16, device=dev)

    def mlp_fp8_chain():
        P.upr_linear_fp8_ex_fwd(layer.h2, 6.0 / 448.0, w1_8, w_scale, prm["b1"], None, u8, 6.0 / 448.0, P.UPR_ACT_SILU, stream)
        P.upr_linear_fp8_ex_fwd(u8, 6.0 / 448.0, w2_8, w2_scale, prm["b2"], x, y8, 1.0, P.UPR_ACT_NONE, stream)

    def mlp_bf16():
        P.upr_linear_fwd(layer.h2, prm["w1"], prm["b1"], layer.u, P.UPR_ACT_SILU, stream)
        P.upr_linear_residual_fwd(layer.u, prm["w2"], prm["b2"], x, y8, P.UPR_ACT_NONE, stream)
    mlp_chain_ms = time_it(mlp_fp8_chain)
    mlp_bf16_ms = time_it(mlp_bf16)
    down_fp8q = time_it(lambda: P.upr_linear_fp8_ex_fwd(u8, 6.0 / 448.0, w2_8, w2_scale, prm["b2"], x, y8, 1.0,
                                                        P.UPR_ACT_NONE, stream))
    # the whole decode layer with the MLP as an FP8 chain (LN2 -> E4M3, up -> E4M3, down -> bf16 + residual),
    # timed alternately with the bf16 layer so that both see the same clocks
    layer8 = pl.RankingDecodeLayer(attn1, D, hidden, prm, fp8_mlp={
        "w1_8": w1_8, "w1_scale": w_scale, "w2_8": w2_8, "w2_scale": w2_scale, "h_scale": 5.0 / 448.0, "u_scale": 6.0 / 448.0})
    ms8 = min(time_it(lambda: layer8(x, stream=stream)) for _ in range(2))
    ms16 = time_it(lambda: layer(x, stream=stream))
    fl_up = 2.0 * M * D * hidden
    gemm_flops = 2.0 * M * D * (4 * D + 2 * hidden)
    attn_flops = (w.flops / w.n_layers) + 4.0 * w.d * M * w.H      # one layer's pairs + the self pair
    return {"ms": ms, "candidates_per_s": M / (ms * 1e-3), "launches": layer.launches, "D_model": D, "mlp_hidden": hidden,
            "gemm_flops": gemm_flops, "attn_flops": attn_flops, "tflops": (gemm_flops + attn_flops) / (ms * 1e-3) / 1e12,
            "mlp_up_bf16_ms": up_bf16, "mlp_up_bf16_tflops": fl_up / (up_bf16 * 1e-3) / 1e12,
            "mlp_up_fp8_ms": up_fp8, "mlp_up_fp8_tflops": fl_up / (up_fp8 * 1e-3) / 1e12,
            "mlp_down_fp8_e4m3_in_ms": down_fp8q, "mlp_down_fp8_e4m3_in_tflops": fl_up / (down_fp8q * 1e-3) / 1e12,
            "mlp_bf16_ms": mlp_bf16_ms, "mlp_bf16_tflops": 2 * fl_up / (mlp_bf16_ms * 1e-3) / 1e12,
            "mlp_fp8_chain_ms": mlp_chain_ms, "mlp_fp8_chain_tflops": 2 * fl_up / (mlp_chain_ms * 1e-3) / 1e12,
            "fp8_mlp_layer_ms": ms8, "bf16_layer_again_ms": ms16, "fp8_mlp_layer_candidates_per_s": M / (ms8 * 1e-3),
            "fp8_mlp_layer_tflops": (gemm_flops + attn_flops) / (ms8 * 1e-3) / 1e12}


def prefill_leg(P, pl, w, pool_shape, slots_host, stream, dev, ev, iters=5):
    """SURVEY 8(f)2, second half, timed: the history prefill of ONE layer over the workload's histories (PAPER.md:138,
    198, 202) -- K / V projections of the history tokens written straight into the pool layout [1,S,H,n,D] by the GEMM's
    epilogue, the Q projection, and the causal O(n^2) self-attention reading those slots in place (pair kernel,
    causal = 1).  Own pools (the workload's are not touched); synthetic weights; C-ABI calls only."""
    import math
    _, S_slots, H, n_max, d = pool_shape
    D = H * d
    L = w.seq_lens.astype(np.int64)
    M = int(L.sum())
    x = S.normal_bf16(w.seed, "pf_x", (M, D), dev)

    def wgt(tag):
        return (S.normal_bf16(w.seed, tag, (D, D), dev).float() / math.sqrt(D)).to(torch.bfloat16)
    wq, wk, wv = wgt("pf_wq"), wgt("pf_wk"), wgt("pf_wv")
    tok_slot = torch.from_numpy(np.repeat(np.asarray(slots_host, dtype=np.int32), L)).to(dev)
    tok_pos = torch.from_numpy(np.concatenate([np.arange(n, dtype=np.int32) for n in L])).to(dev)
    kp = torch.zeros((1, S_slots, H, n_max, d), dtype=torch.bfloat16, device=dev)
    vp = torch.zeros_like(kp)
    qh = torch.empty((M, D), dtype=torch.bfloat16, device=dev)
    co = np.concatenate([[0], np.cumsum(L)]).astype(np.int32)
    view = pl.PoolView.of(kp, vp, torch.as_tensor(np.asarray(slots_host, dtype=np.int32), device=dev), w.seq_lens)
    attn = pl.CrossAttention(view, co, P.UPR_BF16, causal=True)
    e = [ev() for _ in range(3)]

    def once(record=False):
        if record:
            e[0].record(stream)
        P.upr_kv_project_into_pool(x, wk, None, kp, tok_slot, tok_pos, 0, stream)
        P.upr_kv_project_into_pool(x, wv, None, vp, tok_slot, tok_pos, 0, stream)
        P.upr_linear_fwd(x, wq, None, qh, P.UPR_ACT_NONE, stream)
        if record:
            e[1].record(stream)
        attn(qh.view(1, M, H, d), stream=stream)
        if record:
            e[2].record(stream)
    once(); once()
    torch.cuda.synchronize()
    proj_ms, attn_ms = [], []
    for _ in range(iters):
        once(record=True)
        torch.cuda.synchronize()
        proj_ms.append(e[0].elapsed_time(e[1]))
        attn_ms.append(e[1].elapsed_time(e[2]))
    pm, am = float(np.mean(proj_ms)), float(np.mean(attn_ms))
    pairs = float((L * (L + 1) // 2).sum())
    attn_flops = 4.0 * d * H * pairs                 # the visible (query, key) pairs only: QK^T and PV
    proj_flops = 3 * 2.0 * M * D * D
    return {"layers": 1, "history_tokens": M, "D_model": D, "proj_ms": pm, "attn_ms": am, "ms": pm + am,
            "history_tokens_per_s": M / ((pm + am) * 1e-3), "visible_pairs": pairs,
            "attn_flops_visible": attn_flops, "attn_tflops_visible": attn_flops / (am * 1e-3) / 1e12,
            "proj_tflops": proj_flops / (pm * 1e-3) / 1e12, "kernel": P.upr_last_attn_kernel(),
            "note": "causal tiles on the diagonal are half masked: issued MMA flops exceed the visible-pair count"}


# ----------------------------------------------------------------------------- CUDA arm
def run_ours(args):
    import paper_2606_00422_b200 as P
    from paper_2606_00422_b200 import pipeline as pl

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist_
        dist_.init_process_group("nccl", device_id=dev)
        dist = dist_

    w = rank_workload(args.config, rank)
    kv_id, q_id = pl.DTYPE_ID[w.kv_dtype], pl.DTYPE_ID[w.q_dtype]
    # ---- device-resident inputs (the pool is GPU-resident by design)
    q = S.gen_queries(w, "q", dev)
    k_self = S.gen_queries(w, "k_self", dev) if w.self_term else None
    v_self = S.gen_queries(w, "v_self", dev) if w.self_term else None
    k_pool, v_pool = S.gen_pool(w, "k_pool", dev), S.gen_pool(w, "v_pool", dev)
    slots = torch.as_tensor(S.slot_ids(w), device=dev)
    # K/V source: bf16 workloads read the pool IN PLACE (zero copy: the slot copy of PAPER.md:204 is gone
    # from the path); FP8 / fp32 caches need the pack (quantise / widen) and keep it in the step.
    zero_copy = (args.kv_source == "pool") or (args.kv_source == "auto" and w.kv_dtype == "bf16")
    if zero_copy and w.kv_dtype != "bf16":
        raise SystemExit("--kv-source pool needs a bf16 workload (the pool is bf16)")
    cache = pl.alloc_cache(w.seq_lens, w.H, w.d, w.n_layers, kv_id, dev)
    kern = {"auto": P.UPR_KERNEL_AUTO, "single": P.UPR_KERNEL_SINGLE, "pair": P.UPR_KERNEL_PAIR}[args.kernel]
    attn_packed = pl.CrossAttention(cache, w.cand_offsets, q_id, num_splits=0, kernel=kern)
    view = pl.PoolView.of(k_pool, v_pool, slots, w.seq_lens)
    attn = pl.CrossAttention(view, w.cand_offsets, q_id, num_splits=0, kernel=kern) if zero_copy else attn_packed
    stream = torch.cuda.current_stream()
    ev = lambda: torch.cuda.Event(enable_timing=True)  # noqa: E731

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(attn_obj, packed: bool, steps: int, sample_clocks: bool):
        """W warm-ups, then `steps` timed steps with per-kernel events; returns a dict."""
        def one(marks=None):
            n = 0
            if marks:
                marks[0].record(stream)
            # a0: layout is integer-only host work, redone every step like a new batch would
            P.upr_kv_cache_layout(w.seq_lens, w.H, w.d, w.n_layers, kv_id)
            if packed:
                pl.pack_cache(cache, k_pool, v_pool, slots, stream)           # a1
                n += P.upr_last_launch_count()
            if marks:
                marks[1].record(stream)
            attn_obj(q, k_self, v_self, stream=stream)                        # a2-a8
            n += P.upr_last_launch_count()
            if marks:
                marks[2].record(stream)
            return n
        for _ in range(max(args.warmup, 3)):
            one()
        barrier()
        e_start, e_end = ev(), ev()
        marks = [(ev(), ev(), ev()) for _ in range(steps)]
        sampler = ClockSampler(local_rank) if sample_clocks else None
        if sampler:
            sampler.start()
        n_launch = 0
        barrier()
        e_start.record(stream)
        for i in range(steps):
            n_launch += one(marks[i])
        e_end.record(stream)
        barrier()
        clocks = sampler.stop() if sampler else None
        if clocks is not None:
            # what NVML does not show: the clock the SMs really ran at under the attention kernel, from the two
            # counters CTA 0 of the last launch left in the workspace (include/upr.h: bytes [64, 80))
            cyc, ns = (int(x) for x in attn_obj.workspace[64:80].view(torch.int64).tolist())
            if ns > 0:
                clocks["sm_mhz_in_kernel"] = round(1e3 * cyc / ns, 1)
                clocks["in_kernel_how"] = ("clock64 / %globaltimer over the last attention launch (CTA 0); the SM clock "
                                           "follows the tensor-pipe duty cycle, NVML's clocks.sm does not show it")
        return {"total_ms": e_start.elapsed_time(e_end), "clocks": clocks, "launches": n_launch,
                "pack_ms": float(np.mean([a.elapsed_time(b) for a, b, c in marks])),
                "attn_ms": float(np.mean([b.elapsed_time(c) for a, b, c in marks]))}

    main = timed(attn, not zero_copy, args.steps, True)
    attn_kernel_name = P.upr_last_attn_kernel()
    clocks, total_ms, pack_ms, attn_ms = main["clocks"], main["total_ms"], main["pack_ms"], main["attn_ms"]
    launches = [main["launches"]]
    gpu_launches = launches[0]
    ms_step, units = aggregate_over_ranks(total_ms / args.steps, w.total_q, dist)
    value = units / (ms_step * 1e-3)
    # the other variant of the same step (pack + attention over the packed cache), same run, for comparison
    other = None
    if zero_copy and not args.skip_packed_variant:
        o = timed(attn_packed, True, args.steps, False)
        o_ms, _ = aggregate_over_ranks(o["total_ms"] / args.steps, w.total_q, dist)
        other = {"step": "layout + pack(pool->cache) + cross-attention", "ms_per_step": o_ms,
                 "value": units / (o_ms * 1e-3), "pack_ms": o["pack_ms"], "attn_ms": o["attn_ms"]}

    # ---- end-to-end through the public API with HOST buffers (q in, out back), every step.
    # The copies are per layer on their own streams, so layer l+1's queries travel up while layer
    # l is computed and layer l's scores travel back while the next layers run (PCIe is full
    # duplex); every byte of the step's input and output still crosses inside the timed region.
    import dataclasses as _dc
    q_host = q.cpu().pin_memory()
    out_host = torch.empty(attn.out.shape, dtype=torch.float32).pin_memory()
    sl_host = torch.as_tensor(w.seq_lens).pin_memory()
    co_host = torch.as_tensor(w.cand_offsets).pin_memory()
    q_dev2 = torch.empty_like(q)
    e2e_steps = max(1, min(args.steps, 5))
    s_h2d, s_d2h = torch.cuda.Stream(device=dev), torch.cuda.Stream(device=dev)
    lay1, _ = P.upr_kv_cache_layout(w.seq_lens, w.H, w.d, 1, kv_id)
    lstride = int(cache.layout.layer_stride_bytes)
    layer_attn = []
    for l in range(w.n_layers):
        if zero_copy:
            sub = _dc.replace(view, k_pool=k_pool[l:l + 1], v_pool=v_pool[l:l + 1])
        else:
            sub = _dc.replace(cache, layout=lay1,
                              k_cache=cache.k_cache[l * lstride: l * lstride + lay1.bytes_cache],
                              v_cache=cache.v_cache[l * lstride: l * lstride + lay1.bytes_cache],
                              k_scale=None if cache.k_scale is None else cache.k_scale[l * w.H:(l + 1) * w.H],
                              v_scale=None if cache.v_scale is None else cache.v_scale[l * w.H:(l + 1) * w.H])
        layer_attn.append(pl.CrossAttention(sub, w.cand_offsets, q_id, num_splits=0, kernel=kern))
    seq_dev = view.seq_lens if zero_copy else cache.seq_lens
    ev_h = [ev() for _ in range(w.n_layers)]
    ev_c = [ev() for _ in range(w.n_layers)]

    def e2e_step():
        s_h2d.wait_stream(stream)                     # the previous step is done with q_dev2
        with torch.cuda.stream(s_h2d):
            for l in range(w.n_layers):
                q_dev2[l].copy_(q_host[l], non_blocking=True)
                ev_h[l].record(s_h2d)
        seq_dev.copy_(sl_host, non_blocking=True)
        for la in layer_attn:
            la.cand_offsets.copy_(co_host, non_blocking=True)
        P.upr_kv_cache_layout(w.seq_lens, w.H, w.d, w.n_layers, kv_id)            # a0
        if not zero_copy:
            pl.pack_cache(cache, k_pool, v_pool, slots, stream)                   # a1
            launches[0] += P.upr_last_launch_count()
        for l in range(w.n_layers):
            stream.wait_event(ev_h[l])
            out_l = layer_attn[l](q_dev2[l:l + 1],                                # a2-a8, layer l
                                  None if k_self is None else k_self[l:l + 1],
                                  None if v_self is None else v_self[l:l + 1], stream=stream)
            launches[0] += P.upr_last_launch_count()
            ev_c[l].record(stream)
            s_d2h.wait_event(ev_c[l])
            with torch.cuda.stream(s_d2h):
                out_host[l].copy_(out_l[0], non_blocking=True)
        stream.wait_stream(s_d2h)                     # the step ends when its result is on the host
    e2e_step()
    barrier()
    e0, e1 = ev(), ev()
    e0.record(stream)
    for _ in range(e2e_steps):
        e2e_step()
    e1.record(stream)
    barrier()
    e2e_ms, _ = aggregate_over_ranks(e0.elapsed_time(e1) / e2e_steps, w.total_q, dist)
    h2d = q_host.numel() * q_host.element_size() + sl_host.numel() * 4 + co_host.numel() * 4 * w.n_layers
    d2h = out_host.numel() * 4
    # the host copy of the result must be the device result (checked outside the timed region)
    torch.cuda.synchronize()
    assert torch.equal(out_host[0, :64], layer_attn[0].out[0, :64].cpu()), "e2e result did not reach the host"

    # ---- the rest of the ranking pass on the device, reported beside the hot path: the
    # last layer's attention output -> out-projection (tcgen05 GEMM, fp32 rows converted in-kernel) -> stacked
    # first layers of the per-action heads (GEMM + SiLU) -> probabilities -> utility -> per-user top-K.  With it
    # the attention output never leaves the chip: only K indices per user go back to the host.
    tail = None
    if not args.skip_tail and w.q_dtype == "bf16":
        tail = ranking_tail(P, w, attn, q, k_self, v_self, q_host, stream, dev, ev)
        if w.kv_dtype == "bf16" and w.d == 128:
            tail["decode_layer"] = decode_layer_leg(P, pl, w, k_pool, v_pool, slots, stream, dev, ev)
            if int(w.seq_lens.sum()) * w.H * w.d <= (1 << 29):      # bounded: <= 1 GiB of bf16 activations
                tail["prefill"] = prefill_leg(P, pl, w, tuple(k_pool.shape), S.slot_ids(w), stream, dev, ev)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (attention): a dense contraction -> tensor peak
    peaks = measured_peaks()
    flops = w.flops
    tflops = flops / (attn_ms * 1e-3) / 1e12
    t_flop = flops / (peaks["bf16_tflops"] * 1e12)
    t_mem = w.kv_bytes / (peaks["hbm_gbs"] * 1e9)
    roof_ms = 1e3 * max(t_flop, t_mem)
    # ncu counters cannot be read from inside an unprofiled run: the DRAM bytes of the ncu capture of this kernel on
    # this workload are recorded in profiles/r2n_traffic.json (None when there is no capture for it)
    traffic, traffic_source = None, "no ncu capture recorded for this workload"
    try:
        rec = json.load(open(os.path.join(ROOT, "profiles", "r2n_traffic.json"))).get(w.name)
        if rec and rec["kernel"] == attn_kernel_name:
            traffic, traffic_source = rec["dram_read"] + rec["dram_write"], rec["source"] + " (ncu dram__bytes_read.sum + dram__bytes_write.sum, one launch)"
    except OSError:
        pass
    # the bound decides the unit: a tensor-bound workload reports TFLOP/s against the bf16 peak, an HBM-bound one
    # (S1, config 1) its K/V bytes per second against the measured copy bandwidth
    kv_gbs = w.kv_bytes / (attn_ms * 1e-3) / 1e9
    tensor_bound = t_flop >= t_mem
    roofline = {"bound": "tensor" if tensor_bound else "hbm", "kernel": attn_kernel_name,
                "achieved": tflops if tensor_bound else kv_gbs,
                "peak": peaks["bf16_tflops"] if tensor_bound else peaks["hbm_gbs"],
                "unit": "TFLOP/s" if tensor_bound else "GB/s",
                "frac": tflops / peaks["bf16_tflops"] if tensor_bound else kv_gbs / peaks["hbm_gbs"],
                "tflops": tflops, "frac_of_tensor_peak": tflops / peaks["bf16_tflops"],
                "traffic": traffic, "traffic_source": traffic_source,
                "traffic_algorithmic": w.kv_bytes + 6 * w.total_q * w.H * w.d * w.n_layers,
                "peak_source": peaks["source"] + (" (burst cuBLAS bf16)" if tensor_bound else " (device copy bandwidth)"),
                "frac_of_sustained": tflops / peaks["bf16_tflops_sustained"],
                "kernel_ms": attn_ms, "roofline_ms": roof_ms, "frac_of_roofline_time": roof_ms / attn_ms,
                "flops_per_launch": flops, "kv_bytes_per_launch": w.kv_bytes,
                "kv_gbs": kv_gbs}
    # pack: read the valid pool rows (bf16) + write the cache rows; FP8 reads the pool twice (amax, quantise)
    pool_bytes = int(w.seq_lens.astype(np.int64).sum()) * w.H * w.d * w.n_layers * 2 * 2
    pack_bytes = pool_bytes * (2 if w.kv_dtype == "fp8" else 1) + w.kv_bytes
    extra = {"pack_ms": 0.0 if zero_copy else pack_ms, "attn_ms": attn_ms,
             "pack_gbs": None if zero_copy else pack_bytes / (pack_ms * 1e-3) / 1e9,
             "attn_candidates_per_s": w.total_q / (attn_ms * 1e-3), "splits": attn.splits,
             "kv_source": "pool (zero copy)" if zero_copy else "packed decode cache",
             "packed_variant": None if other is None else dict(
                 other, pack_gbs=pack_bytes / (other["pack_ms"] * 1e-3) / 1e9),
             "ranking_tail": tail}

    # ---- CPU baseline: the oracle as it stands, bounded sample, host cores of this box
    cpu_baseline = None
    if not args.skip_cpu_baseline:
        import oracle
        users = oracle_sample_users(w, 15.0)
        t_cpu, cands = oracle_step(w, users)
        sample = f"first {users} of {w.B} users of {w.name}, all layers and heads, pack + attention, {t_cpu:.1f} s"
        cpu_baseline = {"value": cands / t_cpu, "unit": "candidates/s", "cores": oracle.num_threads(),
                        "kind": "oracle", "sample": sample}

    line = {"metric": METRIC, "value": value, "unit": "candidates/s", "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "bf16" if w.kv_dtype != "f32" else "f32", "data": "synthetic",
            "config": {"workload": w.name, "B": w.B, "H": w.H, "d": w.d, "layers": w.n_layers,
                       "total_candidates": w.total_q, "sum_history": int(w.seq_lens.sum()),
                       "kv_dtype": w.kv_dtype, "self_term": w.self_term,
                       "step": ("layout + cross-attention reading the pool in place (zero copy, no slot copy), all "
                                "layers" if zero_copy else "layout + pack(pool->cache) + cross-attention, all layers"),
                       "l2": "inputs larger than L2 (K/V %.1f GB per step)" % (w.kv_bytes / 1e9),
                       "parallelism": "users sharded by rank, no collective" if world > 1 else "single GPU"},
            "clocks": clocks, "gpu_launches": gpu_launches,
            "e2e": {"value": units / (e2e_ms * 1e-3), "unit": "candidates/s", "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h, "ms_per_step": e2e_ms, "steps": e2e_steps},
            "roofline": roofline, "cpu_baseline": cpu_baseline, "detail": extra}
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="3")
    ap.add_argument("--kv-source", default="auto", choices=["auto", "pool", "packed"],
                    help="auto: bf16 workloads read the pool in place (zero copy), FP8/fp32 pack first")
    ap.add_argument("--kernel", default="auto", choices=["auto", "single", "pair"],
                    help="attention kernel: the library's choice, or force the 1-CTA / CTA-pair kernel (A/B runs)")
    ap.add_argument("--skip-packed-variant", action="store_true",
                    help="leave out the secondary pack + attention leg of a zero-copy run")
    ap.add_argument("--skip-tail", action="store_true", help="leave out the ranking-tail legs (detail.ranking_tail)")
    ap.add_argument("--skip-cpu-baseline", action="store_true",
                    help="leave out the oracle timing leg (used for the ncu captures under profiles/)")
    args = ap.parse_args()
    args.config = int(args.config) if args.config.isdigit() else args.config
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
