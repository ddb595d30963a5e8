"""GPU parity for the decode-layer tail and the ranking consumer: the tcgen05
linear layer, the per-action head utility, the per-user top-K, and the cross-process pool (CUDA IPC).
Oracle: oracle.linear / action_utility / topk_per_user (plain fp64 definitions, pinned in
tests/test_oracle_tail_pins.py) on the same seeded inputs.

Tolerances (T3): operands are bf16 values (exact in fp64), products are accumulated in
fp32 over K terms of magnitude ~|x||w|: relative error ~ sqrt(K) 2^-24 -- negligible; a bf16 OUTPUT adds one
rounding, 2^-9 relative; fp32 x rows are rounded to bf16 on the way into the MMA (2^-9 relative per element,
independent: ~2^-9 |y| / sqrt(K) ... bounded here by 2^-8 max|y|)."""
import os
import subprocess
import sys

import numpy as np
import pytest
import torch

import oracle
import upr_synth as S

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def P():
    import paper_2606_00422_b200 as pkg
    assert torch.cuda.is_available()
    return pkg


def f64(t):
    return t.detach().cpu().to(torch.float64).numpy()


def weights(seed, tag, N, K, dev):
    """bf16 weights ~ N(0, 1/K) (unit-variance outputs for unit-variance inputs)."""
    return (S.normal_bf16(seed, tag, (N, K), dev).float() / np.sqrt(K)).to(torch.bfloat16)


LINEAR_CASES = [
    # M, N, K, x dtype, y dtype, act, bias
    (128, 128, 64, "bf16", "f32", 0, False),
    (1, 8, 64, "bf16", "f32", 0, True),
    (300, 136, 192, "bf16", "bf16", 1, True),      # ragged M, N not a multiple of the tile, SiLU
    (517, 1024, 1024, "bf16", "bf16", 0, False),   # the out-projection shape (H d = D_model = 1024)
    (517, 1024, 1024, "f32", "bf16", 0, True),     # fp32 activations (the attention output) converted in-kernel
    (130, 264, 128, "f32", "f32", 2, True),
    (4099, 384, 256, "bf16", "f32", 1, False),     # more tiles than SMs
    # enough 256 x 256 tiles for every SM pair: the CTA-pair kernel (cta_group::2) takes these
    (9500, 640, 512, "bf16", "bf16", 1, True),     # ragged M, N = 2.5 tiles
    (9500, 640, 512, "f32", "f32", 0, True),       # fp32 x: converters in both CTAs
    (19001, 256, 128, "bf16", "f32", 2, False),    # a single N tile, two k-steps
]


@pytest.mark.parametrize("case", LINEAR_CASES, ids=[f"M{c[0]}_N{c[1]}_K{c[2]}_{c[3]}_{c[4]}_act{c[5]}" for c in LINEAR_CASES])
def test_linear_matches_oracle(P, case):
    M, N, K, xdt, ydt, act, has_bias = case
    dev = "cuda"
    x = S.normal_bf16(11, "x", (M, K), dev)
    if xdt == "f32":
        x = S.normal_f32(11, "x32", (M, K)).to(dev)
    w = weights(12, "w", N, K, dev)
    b = (S.normal_bf16(13, "b", (N,), dev).float() * 0.5) if has_bias else None
    y = torch.full((M, N), float("nan"), dtype=torch.float32 if ydt == "f32" else torch.bfloat16, device=dev)
    P.upr_linear_fwd(x, w, b, y, act)
    torch.cuda.synchronize()
    assert P.upr_last_launch_count() == 1
    want = oracle.linear(f64(x), f64(w), None if b is None else f64(b), act=act)
    got = f64(y)
    assert np.isfinite(got).all()
    tol = 2e-4 * max(1.0, np.abs(want).max())
    if xdt == "f32":
        tol += 2.0 ** -8 * np.abs(want).max()
    if ydt == "bf16":
        tol += 2.0 ** -8 * np.abs(want).max()
    err = np.abs(got - want).max()
    print(f"max-abs {err:.2e} (tol {tol:.2e}, max|y| {np.abs(want).max():.2f})")
    assert err <= tol


def test_linear_rejects_unsupported(P):
    x = torch.zeros((4, 96), dtype=torch.bfloat16, device="cuda")
    w = torch.zeros((8, 96), dtype=torch.bfloat16, device="cuda")
    y = torch.zeros((4, 8), dtype=torch.float32, device="cuda")
    with pytest.raises(P.UprError) as e:     # K not a multiple of 64
        P.upr_linear_fwd(x, w, None, y)
    assert e.value.status == 2


def test_prefill_writes_kv_into_the_pool_layout_and_attends_in_place(P):
    """history tokens -> K / V projections written STRAIGHT into the pool [L,S,H,n,D] by the GEMM's
    epilogue (no [M, H d] intermediate, no scatter pass) -> causal attention reads the slots in place.
    Checked: (i) the written rows against the oracle's linear layer (one bf16 rounding), every other pool
    element untouched bit for bit; (ii) the causal attention over the pool the GPU wrote against the oracle on
    the oracle's own projections (K / V rounded to bf16 as the pool stores them)."""
    from paper_2606_00422_b200 import pipeline as pl
    dev = "cuda"
    H, d, D, S_slots, n_max, layers = 2, 128, 256, 5, 200, 2
    L = np.array([150, 0, 37, 200], dtype=np.int32)
    slots_h = np.array([3, 0, 4, 1], dtype=np.int32)
    M = int(L.sum())
    x = S.normal_bf16(31, "x_hist", (M, D), dev)
    wk, wv, wq = weights(32, "wk", H * d, D, dev), weights(33, "wv", H * d, D, dev), weights(34, "wq", H * d, D, dev)
    tok_slot = torch.from_numpy(np.repeat(slots_h, L).astype(np.int32)).to(dev)
    tok_pos = torch.from_numpy(np.concatenate([np.arange(n) for n in L]).astype(np.int32)).to(dev)
    sentinel = S.normal_bf16(35, "stale", (layers, S_slots, H, n_max, d), dev)      # stale K/V of earlier requests
    k_pool, v_pool = sentinel.clone(), sentinel.clone()
    layer = 1
    P.upr_kv_project_into_pool(x, wk, None, k_pool, tok_slot, tok_pos, layer)
    P.upr_kv_project_into_pool(x, wv, None, v_pool, tok_slot, tok_pos, layer)
    q = torch.empty((M, H * d), dtype=torch.bfloat16, device=dev)
    P.upr_linear_fwd(x, wq, None, q, P.UPR_ACT_NONE)
    torch.cuda.synchronize()
    k_want, v_want = oracle.linear(f64(x), f64(wk)), oracle.linear(f64(x), f64(wv))
    written = torch.zeros((layers, S_slots, H, n_max), dtype=torch.bool)
    off = np.concatenate([[0], np.cumsum(L)])
    for b in range(len(L)):
        for h in range(H):
            got_k = f64(k_pool[layer, slots_h[b], h, : L[b]])
            got_v = f64(v_pool[layer, slots_h[b], h, : L[b]])
            wk_ = k_want[off[b]:off[b + 1], h * d:(h + 1) * d]
            wv_ = v_want[off[b]:off[b + 1], h * d:(h + 1) * d]
            if L[b]:
                assert np.abs(got_k - wk_).max() <= 2.0 ** -8 * max(1.0, np.abs(wk_).max())
                assert np.abs(got_v - wv_).max() <= 2.0 ** -8 * max(1.0, np.abs(wv_).max())
            written[layer, slots_h[b], h, : L[b]] = True
    untouched = ~written.to(dev)
    assert torch.equal(k_pool[untouched], sentinel[untouched]) and torch.equal(v_pool[untouched], sentinel[untouched])
    # causal attention over the slots the GPU just wrote, in place
    co = np.concatenate([[0], np.cumsum(L)]).astype(np.int32)
    view = pl.PoolView.of(k_pool[layer:layer + 1], v_pool[layer:layer + 1], torch.from_numpy(slots_h).to(dev), L)
    attn = pl.CrossAttention(view, co, P.UPR_BF16, causal=True)
    out = attn(q.view(1, M, H, d)).cpu().numpy()[0]
    torch.cuda.synchronize()
    q_want = oracle.linear(f64(x), f64(wq))
    def r16(a):   # what a bf16 store keeps of an fp64 value (torch's RNE cast: a library routine)
        return torch.from_numpy(a).to(torch.bfloat16).to(torch.float64).numpy()
    worst = 0.0
    for b in range(len(L)):
        if L[b] == 0:
            continue
        for h in range(H):
            sl = slice(off[b], off[b + 1])
            want = oracle.full_sequence_attention(r16(q_want[sl, h * d:(h + 1) * d]), r16(k_want[sl, h * d:(h + 1) * d]),
                                                  r16(v_want[sl, h * d:(h + 1) * d]), int(L[b]), 0, False)
            worst = max(worst, float(np.abs(out[sl, h] - want).max()))
    print(f"prefill chain max-abs {worst:.2e}")
    # q, K, V each carry one bf16 rounding whose tie-breaks may differ from the oracle's by one ulp (2^-8 relative):
    # logits move by ~2^-8 |q||k| / sqrt(d) ~ 4e-3, outputs by a few 1e-3
    assert worst <= 1e-2


def test_layernorm_and_residual_epilogue_match_oracle(P):
    dev = "cuda"
    M, D = 333, 1024
    x = (S.normal_bf16(41, "x", (M, D), dev).float() * 2.0 + 0.5).to(torch.bfloat16)
    g = 1.0 + 0.1 * S.normal_bf16(42, "g", (D,), dev).float()
    b = 0.1 * S.normal_bf16(43, "b", (D,), dev).float()
    y = torch.empty_like(x)
    P.upr_layernorm_fwd(x, g, b, y)
    torch.cuda.synchronize()
    want = oracle.layernorm(f64(x), f64(g), f64(b))
    assert np.abs(f64(y) - want).max() <= 2.0 ** -8 * np.abs(want).max()          # one bf16 rounding of the output
    # residual epilogue: y = x W^T + r
    w = weights(44, "w", 256, D, dev)
    r = S.normal_bf16(45, "r", (M, 256), dev)
    z = torch.empty((M, 256), dtype=torch.bfloat16, device=dev)
    P.upr_linear_residual_fwd(x, w, None, r, z)
    torch.cuda.synchronize()
    want = oracle.linear(f64(x), f64(w)) + f64(r)
    assert np.abs(f64(z) - want).max() <= 2.0 ** -8 * np.abs(want).max() + 1e-3


def test_one_ranking_decode_layer_matches_the_oracle_chain(P):
    """a candidate token through a whole decode layer without leaving the chip -- LN, Q / self-K,V
    projections, cross-attention over the cached history (+ own key/value), out-projection + residual, LN, MLP
    (SiLU) + residual -- against the same chain of oracle functions in fp64.  The oracle rounds to bf16 exactly
    where the GPU stores bf16 (torch's cast as the library routine), so what is compared is the kernels'
    arithmetic, not the storage format."""
    from paper_2606_00422_b200 import pipeline as pl
    dev = "cuda"
    H, d, hidden = 2, 128, 512
    D = H * d
    L, C = [300, 64, 0, 129], [130, 17, 5, 200]
    w = S.custom_workload("layer", 51, L, C, H, d, 1, self_term=True)
    M = w.total_q
    k_pool, v_pool = S.gen_pool(w, "k_pool", dev), S.gen_pool(w, "v_pool", dev)
    slots_h = S.slot_ids(w)
    view = pl.PoolView.of(k_pool, v_pool, torch.as_tensor(slots_h, device=dev), w.seq_lens)
    attn = pl.CrossAttention(view, w.cand_offsets, P.UPR_BF16, kernel=P.UPR_KERNEL_PAIR)
    prm = {"ln1_g": 1.0 + 0.1 * S.normal_bf16(52, "g1", (D,), dev).float(), "ln1_b": 0.1 * S.normal_bf16(53, "b1", (D,), dev).float(),
           "ln2_g": 1.0 + 0.1 * S.normal_bf16(54, "g2", (D,), dev).float(), "ln2_b": 0.1 * S.normal_bf16(55, "b2", (D,), dev).float(),
           "wq": weights(56, "wq", D, D, dev), "wk": weights(57, "wk", D, D, dev), "wv": weights(58, "wv", D, D, dev),
           "wo": weights(59, "wo", D, D, dev), "w1": weights(60, "w1", hidden, D, dev), "w2": weights(61, "w2", D, hidden, dev),
           "b1": 0.1 * S.normal_bf16(62, "bb1", (hidden,), dev).float(), "b2": 0.1 * S.normal_bf16(63, "bb2", (D,), dev).float()}
    x = S.normal_bf16(64, "x", (M, D), dev)
    layer = pl.RankingDecodeLayer(attn, D, hidden, prm)
    y = layer(x)
    torch.cuda.synchronize()
    assert layer.launches == 10            # 2 LN + 6 GEMM + schedule + attention

    def r16(a):
        return torch.from_numpy(np.ascontiguousarray(a)).to(torch.bfloat16).to(torch.float64).numpy()
    o = {k: f64(v) for k, v in prm.items()}
    xf = f64(x)
    h1 = r16(oracle.layernorm(xf, o["ln1_g"], o["ln1_b"]))
    q, ks, vs = (r16(oracle.linear(h1, o[k])) for k in ("wq", "wk", "wv"))
    a = np.zeros((M, H, d))
    co = w.cand_offsets
    for b in range(w.B):
        if co[b + 1] == co[b]:
            continue
        sl = slice(int(co[b]), int(co[b + 1]))
        for h in range(H):
            K = f64(k_pool[0, slots_h[b], h, : L[b]])
            V = f64(v_pool[0, slots_h[b], h, : L[b]])
            a[sl, h] = oracle.attn_block(q[sl, h * d:(h + 1) * d], K, V, ks[sl, h * d:(h + 1) * d], vs[sl, h * d:(h + 1) * d])
    x2 = r16(oracle.linear(r16(a.reshape(M, D)), o["wo"]) + xf)   # the GEMM rounds the fp32 attention output to bf16 on its way in
    h2 = r16(oracle.layernorm(x2, o["ln2_g"], o["ln2_b"]))
    u = r16(oracle.linear(h2, o["w1"], o["b1"], act=oracle.ACT_SILU))
    want = oracle.linear(u, o["w2"], o["b2"]) + x2
    err = np.abs(f64(y) - want).max()
    print(f"decode layer max-abs {err:.2e} (max|y| {np.abs(want).max():.2f})")
    # nine bf16 stores on the way; a value that sits near a rounding boundary may round the other way on the GPU
    # (2^-8 relative) and that difference propagates through the later GEMMs with unit gain: a few 2^-8 max|y|
    assert err <= 4 * 2.0 ** -8 * np.abs(want).max()



def _codes_agree(got8, want_values_f64, scale, max_differ=5e-3):
    """E4M3 bytes from the GPU against the oracle's quantisation of its own fp64 values: equal except where a value
    sits on a rounding boundary (the GPU decides on its fp32 value), and then one E4M3 step apart at most."""
    code_want = oracle.e4m3_encode((want_values_f64.astype(np.float32) * (np.float32(1.0) / np.float32(scale))).astype(np.float32))
    differ = got8 != code_want
    dec_g, dec_w = oracle.e4m3_decode(got8), oracle.e4m3_decode(code_want)
    step = np.maximum(np.abs(dec_w), 2.0 ** -6) * 2.0 ** -3
    assert differ.mean() < max_differ, differ.mean()
    assert (np.abs(dec_g - dec_w) <= step + 1e-12).all()
    return float(differ.mean())


def test_decode_layer_with_an_fp8_mlp_chain(P):
    """PAPER.md:206 (FP8 linear layers) inside the decode layer: LN2 writes E4M3, up-projection (E4M3 x E4M3, SiLU)
    writes E4M3, down-projection (E4M3 x E4M3) + residual writes bf16.  Each stage is checked against the oracle fed
    the GPU's OWN input bytes of that stage, so every comparison is between the same operands."""
    from paper_2606_00422_b200 import pipeline as pl
    dev = "cuda"
    H, d, hidden = 2, 128, 1024
    D = H * d
    L, C = [300, 64, 0, 129], [700, 17, 5, 600]
    w = S.custom_workload("layer8", 151, L, C, H, d, 1, self_term=True)
    M = w.total_q
    k_pool, v_pool = S.gen_pool(w, "k_pool", dev), S.gen_pool(w, "v_pool", dev)
    view = pl.PoolView.of(k_pool, v_pool, torch.as_tensor(S.slot_ids(w), device=dev), w.seq_lens)
    attn = pl.CrossAttention(view, w.cand_offsets, P.UPR_BF16)
    prm = {"ln1_g": torch.ones(D, device=dev), "ln1_b": torch.zeros(D, device=dev),
           "ln2_g": 1.0 + 0.1 * S.normal_bf16(154, "g2", (D,), dev).float(), "ln2_b": 0.1 * S.normal_bf16(155, "b2", (D,), dev).float(),
           "wq": weights(156, "wq", D, D, dev), "wk": weights(157, "wk", D, D, dev), "wv": weights(158, "wv", D, D, dev),
           "wo": weights(159, "wo", D, D, dev), "w1": weights(160, "w1", hidden, D, dev), "w2": weights(161, "w2", D, hidden, dev),
           "b1": 0.1 * S.normal_bf16(162, "bb1", (hidden,), dev).float(), "b2": 0.1 * S.normal_bf16(163, "bb2", (D,), dev).float()}

    def q8(wt):
        wf = wt.float()
        sc = float(np.float32(wf.abs().max().item()) / np.float32(448.0))
        return (wf * (np.float32(1.0) / np.float32(sc))).to(torch.float8_e4m3fn).view(torch.uint8), sc
    w1_8, w1_s = q8(prm["w1"])
    w2_8, w2_s = q8(prm["w2"])
    f8 = {"w1_8": w1_8, "w1_scale": w1_s, "w2_8": w2_8, "w2_scale": w2_s,
          "h_scale": float(np.float32(5.0) / np.float32(448.0)), "u_scale": float(np.float32(6.0) / np.float32(448.0))}
    x = S.normal_bf16(164, "x", (M, D), dev)
    layer = pl.RankingDecodeLayer(attn, D, hidden, prm, fp8_mlp=f8)
    y = layer(x)
    torch.cuda.synchronize()
    assert layer.launches == 10
    x2 = f64(layer.x2)
    h8, u8 = layer.h2_8.cpu().numpy(), layer.u_8.cpu().numpy()
    d1 = _codes_agree(h8, oracle.layernorm(x2, f64(prm["ln2_g"]), f64(prm["ln2_b"])), f8["h_scale"])
    d2 = _codes_agree(u8, oracle.linear_fp8q(h8, f8["h_scale"], w1_8.cpu().numpy(), w1_s, f64(prm["b1"]), act=oracle.ACT_SILU),
                      f8["u_scale"])
    want = oracle.linear_fp8q(u8, f8["u_scale"], w2_8.cpu().numpy(), w2_s, f64(prm["b2"])) + x2
    err = np.abs(f64(y) - want).max()
    print(f"fp8 mlp: codes differing {d1:.1e} (LN2), {d2:.1e} (up); down-projection max-abs {err:.2e}")
    assert err <= 2.0 ** -8 * max(1.0, np.abs(want).max()) + 2e-4


def test_pair_gemm_residual_and_pool_epilogues(P):
    """The CTA-pair GEMM's residual and pool-addressing epilogues (M large enough for the pair kernel)."""
    dev = "cuda"
    M, D = 19200, 256
    x = S.normal_bf16(71, "x", (M, D), dev)
    w = weights(72, "w", D, D, dev)
    r = S.normal_bf16(73, "r", (M, D), dev)
    z = torch.empty((M, D), dtype=torch.bfloat16, device=dev)
    P.upr_linear_residual_fwd(x, w, None, r, z)
    torch.cuda.synchronize()
    want = oracle.linear(f64(x), f64(w))
    assert np.abs(f64(z) - (want + f64(r))).max() <= 2.0 ** -8 * np.abs(want + f64(r)).max() + 1e-3
    # K projection of 19 200 tokens (96 users x 200 positions) into a pool [1, 100, 2, 200, 128]
    H, d, S_slots, n = 2, 128, 100, 200
    pool = torch.zeros((1, S_slots, H, n, d), dtype=torch.bfloat16, device=dev)
    slot_of_user = np.random.default_rng(3).permutation(S_slots)[:96].astype(np.int32)
    tok_slot = torch.from_numpy(np.repeat(slot_of_user, n)).to(dev)
    tok_pos = torch.from_numpy(np.tile(np.arange(n, dtype=np.int32), 96)).to(dev)
    P.upr_kv_project_into_pool(x, w, None, pool, tok_slot, tok_pos, 0)
    torch.cuda.synchronize()
    got = f64(pool)
    for u in (0, 37, 95):
        for h in range(H):
            blk = want[u * n:(u + 1) * n, h * d:(h + 1) * d]
            assert np.abs(got[0, slot_of_user[u], h] - blk).max() <= 2.0 ** -8 * max(1.0, np.abs(blk).max())
    unused = np.setdiff1d(np.arange(S_slots), slot_of_user)
    assert not got[0, unused].any()


@pytest.mark.parametrize("shape", [(300, 136, 256), (9500, 640, 512), (64, 8, 128)], ids=["ragged", "many_tiles", "tiny"])
def test_linear_fp8_matches_oracle(P, shape):
    """PAPER.md:206 / SURVEY 8(f)1: FP8 E4M3 linear layer with fused scaling (tcgen05 kind::f8f6f4 on CTA pairs): the
    activations are quantised inside the kernel exactly as the oracle does (one fp32 product, RNE, satfinite), the
    weights arrive as E4M3 bytes, so both sides multiply the SAME operands: what differs is fp32 accumulation."""
    M, N, K = shape
    dev = "cuda"
    x = S.normal_bf16(81, "x", (M, K), dev)
    wf = (S.normal_bf16(82, "w", (N, K), dev).float() / np.sqrt(K))
    x_scale = float(np.float32(4.5) / np.float32(448.0))            # a fixed ("delayed") activation scale: clips beyond 4.5 sigma
    w_scale = float(np.float32(wf.abs().max().item()) / np.float32(448.0))
    w8 = (wf * (np.float32(1.0) / np.float32(w_scale))).to(torch.float8_e4m3fn).view(torch.uint8)   # offline weight quantisation
    b = S.normal_bf16(83, "b", (N,), dev).float() * 0.5
    r = S.normal_bf16(84, "r", (M, N), dev)
    y = torch.empty((M, N), dtype=torch.float32, device=dev)
    P.upr_linear_fp8_fwd(x, x_scale, w8, w_scale, b, r, y, P.UPR_ACT_SILU)
    torch.cuda.synchronize()
    want = oracle.linear_fp8(x.float().cpu().numpy(), x_scale, w8.cpu().numpy(), w_scale, f64(b), act=oracle.ACT_SILU) + f64(r)
    err = np.abs(f64(y) - want).max()
    print(f"fp8 linear max-abs {err:.2e} (max|y| {np.abs(want).max():.2f})")
    assert err <= 2e-4 * max(1.0, np.abs(want).max())



def test_fp8_chain_keeps_the_hidden_tensor_in_e4m3(P):
    """MLP up -> down as an FP8 chain (upr_linear_fp8_ex_fwd): the first layer leaves E4M3 bytes, the second reads
    them through TMA.  Layer 1's bytes: the quantisation decision is taken on the GPU's own fp32 value, the oracle's
    on its fp64 value rounded to fp32 -- codes may differ where a value sits on a rounding boundary, by one E4M3 step
    at most, for a small fraction.  Layer 2 is checked against the oracle fed the GPU's OWN bytes (same operands)."""
    M, D, F = 1500, 256, 1024
    dev = "cuda"
    x = S.normal_bf16(91, "x", (M, D), dev)
    w1f = S.normal_bf16(92, "w1", (F, D), dev).float() / np.sqrt(D)
    w2f = S.normal_bf16(93, "w2", (D, F), dev).float() / np.sqrt(F)
    q8 = lambda wf, sc: (wf * (np.float32(1.0) / np.float32(sc))).to(torch.float8_e4m3fn).view(torch.uint8)
    x_scale = float(np.float32(4.5) / np.float32(448.0))
    w1_scale = float(np.float32(w1f.abs().max().item()) / np.float32(448.0))
    w2_scale = float(np.float32(w2f.abs().max().item()) / np.float32(448.0))
    h_scale = float(np.float32(6.0) / np.float32(448.0))           # SiLU outputs of unit-variance pre-activations
    w1, w2 = q8(w1f, w1_scale), q8(w2f, w2_scale)
    b1 = S.normal_bf16(94, "b1", (F,), dev).float() * 0.2
    b2 = S.normal_bf16(95, "b2", (D,), dev).float() * 0.2
    h8 = torch.empty((M, F), dtype=torch.uint8, device=dev)
    y = torch.empty((M, D), dtype=torch.bfloat16, device=dev)
    P.upr_linear_fp8_ex_fwd(x, x_scale, w1, w1_scale, b1, None, h8, h_scale, P.UPR_ACT_SILU)
    assert P.upr_last_launch_count() == 1
    P.upr_linear_fp8_ex_fwd(h8, h_scale, w2, w2_scale, b2, x, y, 1.0, P.UPR_ACT_NONE)
    torch.cuda.synchronize()
    # layer 1
    h_want = oracle.linear_fp8(x.float().cpu().numpy(), x_scale, w1.cpu().numpy(), w1_scale, f64(b1), act=oracle.ACT_SILU)
    code_want = oracle.e4m3_encode((h_want.astype(np.float32) * (np.float32(1.0) / np.float32(h_scale))).astype(np.float32))
    got8 = h8.cpu().numpy()
    differ = got8 != code_want
    dec_g, dec_w = oracle.e4m3_decode(got8), oracle.e4m3_decode(code_want)
    step = np.maximum(np.abs(dec_w), 2.0 ** -6) * 2.0 ** -3        # one E4M3 step at that magnitude (3 mantissa bits)
    assert differ.mean() < 5e-3, differ.mean()
    assert (np.abs(dec_g - dec_w) <= step + 1e-12).all()
    print(f"fp8 chain: {differ.mean():.2e} of layer-1 codes differ (all by <= one step)")
    # layer 2 on the GPU's bytes
    y_want = oracle.linear_fp8q(got8, h_scale, w2.cpu().numpy(), w2_scale, f64(b2)) + f64(x)
    err = np.abs(f64(y) - y_want).max()
    assert err <= 2.0 ** -8 * max(1.0, np.abs(y_want).max()) + 2e-4, err     # bf16 output rounding
    # errors are reported, not hidden
    with pytest.raises(P.UprError):
        P.upr_linear_fp8_ex_fwd(h8, 0.0, w2, w2_scale, b2, None, y, 1.0)


def test_action_heads_and_utility_match_oracle(P):
    """z -> [stacked first layers of the C heads, SiLU] (tcgen05 GEMM) -> logits -> sigmoid -> utility."""
    dev = "cuda"
    M, D, C, Dh = 777, 256, 5, 64
    z = S.normal_bf16(21, "z", (M, D), dev)
    w1 = weights(22, "w1", C * Dh, D, dev)
    b1 = S.normal_bf16(23, "b1", (C * Dh,), dev).float() * 0.1
    w2 = (S.normal_bf16(24, "w2", (C, Dh), dev).float() / np.sqrt(Dh)).contiguous()
    b2 = S.normal_bf16(25, "b2", (C,), dev).float() * 0.1
    wc = torch.tensor([1.0, 0.5, 2.0, 0.25, 1.5], device=dev)
    hid = torch.empty((M, C * Dh), dtype=torch.bfloat16, device=dev)
    probs = torch.empty((M, C), dtype=torch.float32, device=dev)
    util = torch.empty(M, dtype=torch.float32, device=dev)
    P.upr_linear_fwd(z, w1, b1, hid, P.UPR_ACT_SILU)
    P.upr_action_utility(hid, w2, b2, wc, probs, util)
    torch.cuda.synchronize()
    want_p, want_u = oracle.action_utility(f64(z), f64(w1).reshape(C, Dh, D), f64(b1).reshape(C, Dh), f64(w2), f64(b2),
                                           f64(wc))
    ep, eu = np.abs(f64(probs) - want_p).max(), np.abs(f64(util) - want_u).max()
    print(f"probs max-abs {ep:.2e}, utility max-abs {eu:.2e}")
    # hid is rounded to bf16 (2^-9 relative, Dh independent terms): logit error ~ 2^-9 |logit| -> prob error <= 1/4 of it
    assert ep <= 2e-3 and eu <= 2e-3 * float(wc.sum())


def test_topk_matches_oracle_bit_for_bit(P):
    dev = "cuda"
    rng = np.random.default_rng(5)
    counts = np.array([0, 1, 5, 1000, 37, 4096, 129, 0, 2], dtype=np.int64)
    co = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
    util_h = (rng.integers(-50, 50, size=co[-1]) / 16.0).astype(np.float32)     # many exact ties
    util_h[7] = -0.0
    util = torch.from_numpy(util_h).to(dev)
    for K in (1, 10, 300):
        idx = torch.full((len(counts), K), -7, dtype=torch.int32, device=dev)
        cnt = torch.full((len(counts),), -7, dtype=torch.int32, device=dev)
        P.upr_topk_per_user(util, torch.from_numpy(co).to(dev), K, int(counts.max()), idx, cnt)
        torch.cuda.synchronize()
        want_idx, want_cnt = oracle.topk_per_user(util_h, co, K)
        assert np.array_equal(cnt.cpu().numpy(), want_cnt)
        assert np.array_equal(idx.cpu().numpy(), want_idx)
    with pytest.raises(P.UprError) as e:
        P.upr_topk_per_user(util, torch.from_numpy(co).to(dev), 4, 20000, idx, cnt)
    assert e.value.status == 2


_CHILD = r"""
import sys, numpy as np, torch
sys.path.insert(0, {root!r})
import paper_2606_00422_b200 as P
handle = bytes.fromhex(sys.argv[1]); n = int(sys.argv[2])
ptr = P.upr_pool_open(handle)
# wrap the mapped allocation (no copy) and read it; then run the attention on it in place
import ctypes
class _Arr:  # minimal __cuda_array_interface__ holder
    def __init__(self, ptr, n): self.__cuda_array_interface__ = dict(shape=(n,), typestr='<i2', data=(ptr, False), version=3)
t = torch.as_tensor(_Arr(ptr, n), device='cuda')
print('SUM', int(t.to(torch.int64).sum().item()))
del t
P.upr_pool_close(ptr)
"""


def test_pool_crosses_process_boundary_through_cuda_ipc(P, tmp_path):
    """the retrieval process allocates the pool and exports an IPC handle 'to a per-instance
    file'; the ranking process opens it and reads the same physical allocation.  Parent = retrieval replica,
    child = ranking consumer."""
    pool = (torch.arange(0, 50000, device="cuda") % 30011).to(torch.int16)     # stands in for the bf16 pool's bits
    torch.cuda.synchronize()
    handle = P.upr_pool_export(pool)
    (tmp_path / "pool.handle").write_bytes(handle)                             # the per-instance file
    script = tmp_path / "child.py"
    script.write_text(_CHILD.format(root=ROOT))
    r = subprocess.run([sys.executable, str(script), (tmp_path / "pool.handle").read_bytes().hex(), str(pool.numel())],
                       capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    assert f"SUM {int(pool.to(torch.int64).sum().item())}" in r.stdout


def test_slot_ring_round_robin(P):
    ring = P.SlotRing(5)
    assert ring.acquire(3).tolist() == [0, 1, 2]
    assert ring.acquire(4).tolist() == [3, 4, 0, 1]
    with pytest.raises(P.UprError):
        ring.acquire(6)
