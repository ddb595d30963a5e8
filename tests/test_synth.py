"""Host-side checks of the seeded input generators (upr_synth.py)."""
import numpy as np
import torch

import upr_synth as S


def test_torch_hash_matches_scalar_splitmix64():
    key = S.stream_key(1234, "q")
    h = S.hash_u64(key, 5, 64, "cpu").numpy().view(np.uint64)
    want = np.array([S.hash_u64_scalar(key, i) for i in range(5, 69)], dtype=np.uint64)
    assert np.array_equal(h, want)
    # splitmix64 published first outputs for state 0: 0xE220A8397B1DCDAF, 0x6E789E6AA1B965F4
    assert S.splitmix64(0) == 0xE220A8397B1DCDAF
    assert S.splitmix64(S._GAMMA) == 0x6E789E6AA1B965F4


def test_normal_bf16_is_order_independent_and_unit_variance():
    a = S.normal_bf16(7, "k", (1000, 64), chunk=1 << 25)
    b = S.normal_bf16(7, "k", (1000, 64), chunk=777)
    assert torch.equal(a, b)
    x = S.normal_bf16(11, "v", (1 << 20,)).float()
    assert abs(float(x.mean())) < 5e-3 and abs(float(x.var()) - 1.0) < 1e-2
    assert float(x.abs().max()) < 4.5
    assert not torch.equal(S.normal_bf16(11, "k", (64,)), S.normal_bf16(11, "v", (64,)))


def test_workloads_match_baseline_configs():
    w = S.workload(1)
    assert (w.B, w.H, w.d, w.n_layers, w.total_q, w.kv_dtype) == (1, 4, 64, 1, 16, "f32") and w.seq_lens[0] == 256
    w = S.workload(2)
    assert (w.B, w.H, w.d, w.total_q) == (64, 8, 64, 64 * 256)
    assert w.seq_lens.min() >= 128 and w.seq_lens.max() <= 1024
    w = S.workload(3)
    assert (w.B, w.H, w.d, w.n_layers, w.total_q) == (256, 8, 128, 4, 256 * 512)
    assert w.seq_lens.min() >= 512 and w.seq_lens.max() <= 2048
    assert abs(w.flops / 2.749e12 - 1) < 0.1
    w = S.workload(4)
    assert (w.B, w.H, w.d, w.n_layers, w.total_q, w.kv_dtype) == (128, 16, 64, 2, 128000, "fp8")
    assert w.flops == 4 * 64 * 128 * 1000 * 4096 * 16 * 2
    w = S.workload(5)
    assert (w.B, w.H, w.d, w.self_term) == (512, 8, 128, True)
    c = w.cand_counts
    assert c.min() >= 50 and c.max() <= 1000 and w.seq_lens.min() >= 64 and w.seq_lens.max() <= 8192
    # log-uniform: median near sqrt(64*8192) = 724
    assert 400 < np.median(w.seq_lens) < 1300
    assert sorted(S.slot_ids(w).tolist()) == list(range(512))
    small = S.workload(3, users=3)
    assert small.B == 3 and np.array_equal(small.seq_lens, S.workload(3).seq_lens[:3])
