"""Pins for the CPU fp64 oracle (oracle/upr_oracle.c) against what the paper and the
mathematics fix -- none of these re-types the oracle's own formula.  Run with -m "not gpu".

The paper prints no worked numerical example of the attention, so the
pins are closed forms, invariants the paper states (PAPER.md:198 batch-composition
independence; PAPER.md:138 the masked full-sequence formulation and its pair count),
a library special case (torch SDPA in fp64 with an explicit mask) and brute force.
"""
import numpy as np
import pytest
import torch


def rng(seed):
    return np.random.default_rng(seed)


# ----------------------------------------------------------------------- softmax weights
def test_softmax_rows_sum_to_one(oracle):
    r = rng(0)
    for (C, L, d, self_on) in [(3, 7, 8, False), (5, 33, 16, True), (1, 1, 4, True), (4, 200, 64, False)]:
        q, K, V = r.standard_normal((C, d)), r.standard_normal((L, d)), r.standard_normal((L, d))
        ks = r.standard_normal((C, d)) if self_on else None
        vs = r.standard_normal((C, d)) if self_on else None
        _, w = oracle.attn_block(q, K, V, ks, vs, return_weights=True)
        assert np.all(w >= 0)
        np.testing.assert_allclose(w.sum(axis=1), 1.0, rtol=0, atol=1e-14)
        if not self_on:
            assert np.all(w[:, -1] == 0)


def test_one_hot_values_expose_weights(oracle):
    """With V = identity rows (L <= d) the output IS the weight vector."""
    r = rng(1)
    C, L, d = 4, 6, 8
    q, K = r.standard_normal((C, d)), r.standard_normal((L, d))
    V = np.zeros((L, d))
    V[np.arange(L), np.arange(L)] = 1.0
    out, w = oracle.attn_block(q, K, V, return_weights=True)
    np.testing.assert_allclose(out[:, :L], w[:, :L], rtol=0, atol=1e-15)
    # and the weights are the textbook softmax of q.K^T/sqrt(d), computed here independently
    s = (q @ K.T) / np.sqrt(d)
    e = np.exp(s - s.max(axis=1, keepdims=True))
    np.testing.assert_allclose(w[:, :L], e / e.sum(axis=1, keepdims=True), rtol=1e-13, atol=1e-15)


# ----------------------------------------------------------------------- single key / closed forms
def test_single_key_returns_its_value_row(oracle):
    r = rng(2)
    q, K, V = r.standard_normal((5, 16)), r.standard_normal((1, 16)), r.standard_normal((1, 16))
    out = oracle.attn_block(q, K, V)
    assert np.array_equal(out, np.repeat(V, 5, axis=0))


def test_no_history_with_self_returns_vself(oracle):
    r = rng(3)
    q, ks, vs = r.standard_normal((4, 8)), r.standard_normal((4, 8)), r.standard_normal((4, 8))
    out = oracle.attn_block(q, np.zeros((0, 8)), np.zeros((0, 8)), ks, vs)
    assert np.array_equal(out, vs)


def test_no_logits_gives_zeros_not_nan(oracle):
    out = oracle.attn_block(np.ones((3, 8)), np.zeros((0, 8)), np.zeros((0, 8)))
    assert np.array_equal(out, np.zeros((3, 8)))


def test_identical_keys_or_zero_query_give_mean_of_values(oracle):
    r = rng(4)
    L, d = 37, 16
    V = r.standard_normal((L, d))
    K = np.repeat(r.standard_normal((1, d)), L, axis=0)
    out = oracle.attn_block(r.standard_normal((3, d)), K, V)
    np.testing.assert_allclose(out, np.repeat(V.mean(axis=0, keepdims=True), 3, axis=0), rtol=0, atol=1e-14)
    out0 = oracle.attn_block(np.zeros((2, d)), r.standard_normal((L, d)), V)
    np.testing.assert_allclose(out0, np.repeat(V.mean(axis=0, keepdims=True), 2, axis=0), rtol=0, atol=1e-14)


def test_sharp_query_selects_argmax_value_and_is_stable(oracle):
    r = rng(5)
    C, L, d = 6, 50, 16
    q, K, V = r.standard_normal((C, d)), r.standard_normal((L, d)), r.standard_normal((L, d))
    out = oracle.attn_block(q * 1e4, K, V)  # logits ~ 1e4: exp overflows without max-subtraction
    assert np.all(np.isfinite(out))
    best = np.argmax(q @ K.T, axis=1)
    np.testing.assert_allclose(out, V[best], rtol=0, atol=1e-12)


def test_scale_default_is_inverse_sqrt_d(oracle):
    """Two keys, hand-computed: w0 = sigmoid((q.k0 - q.k1)/sqrt(d))."""
    d = 4
    q = np.array([[1.0, 2.0, 0.0, -1.0]])
    K = np.array([[1.0, 0.0, 0.0, 0.0], [0.0, 1.0, 0.0, 0.0]])
    V = np.array([[1.0, 0, 0, 0], [0, 1.0, 0, 0]])
    out = oracle.attn_block(q, K, V)
    w0 = 1.0 / (1.0 + np.exp((2.0 - 1.0) / 2.0))  # s0 = 1/2, s1 = 2/2
    np.testing.assert_allclose(out[0, :2], [w0, 1 - w0], rtol=1e-15)


# ----------------------------------------------------------------------- invariants
def test_candidate_permutation_and_batch_composition(oracle):
    """'each candidate's score is independent of the batch composition'."""
    r = rng(6)
    C, L, d = 9, 40, 16
    q, K, V = r.standard_normal((C, d)), r.standard_normal((L, d)), r.standard_normal((L, d))
    ks, vs = r.standard_normal((C, d)), r.standard_normal((C, d))
    for self_on in (False, True):
        a = (ks, vs) if self_on else (None, None)
        full = oracle.attn_block(q, K, V, *a)
        perm = r.permutation(C)
        pa = (ks[perm], vs[perm]) if self_on else (None, None)
        assert np.array_equal(oracle.attn_block(q[perm], K, V, *pa), full[perm])
        for c in range(C):
            sa = (ks[c:c + 1], vs[c:c + 1]) if self_on else (None, None)
            assert np.array_equal(oracle.attn_block(q[c:c + 1], K, V, *sa), full[c:c + 1])


def test_key_permutation_and_logit_shift_invariance(oracle):
    r = rng(7)
    C, L, d = 4, 60, 8
    q, K, V = r.standard_normal((C, d)), r.standard_normal((L, d)), r.standard_normal((L, d))
    base = oracle.attn_block(q, K, V)
    p = r.permutation(L)
    np.testing.assert_allclose(oracle.attn_block(q, K[p], V[p]), base, rtol=0, atol=1e-13)
    # add the same constant to every logit: append one coordinate, equal on all keys
    q2 = np.concatenate([q, np.full((C, 1), 3.0)], axis=1)
    K2 = np.concatenate([K, np.full((L, 1), 1.7)], axis=1)
    V2 = np.concatenate([V, np.zeros((L, 1))], axis=1)
    out2 = oracle.attn_block(q2, K2, V2, scale=1.0 / np.sqrt(d))
    np.testing.assert_allclose(out2[:, :d], base, rtol=0, atol=1e-13)


def test_same_cache_serves_different_candidate_sets(oracle):
    """candidate-independent history representations cached once."""
    r = rng(8)
    L, d = 30, 8
    K, V = r.standard_normal((L, d)), r.standard_normal((L, d))
    qa, qb = r.standard_normal((3, d)), r.standard_normal((5, d))
    both = oracle.attn_block(np.concatenate([qa, qb]), K, V)
    assert np.array_equal(both[:3], oracle.attn_block(qa, K, V))
    assert np.array_equal(both[3:], oracle.attn_block(qb, K, V))


# ----------------------------------------------------------------------- the paper's masked formulation
@pytest.mark.parametrize("self_flag", [False, True])
def test_equals_masked_full_sequence_attention(oracle, self_flag):
    """full sequence [history || candidates] with the M-FALCON mask; the
    candidate rows must equal the cached-K/V decode path."""
    r = rng(9)
    n, k, d = 23, 7, 16
    xq, xk, xv = (r.standard_normal((n + k, d)) for _ in range(3))
    dense, mask = oracle.full_sequence_attention(xq, xk, xv, n, k, self_flag, return_mask=True)
    cached = oracle.attn_block(xq[n:], xk[:n], xv[:n], xk[n:] if self_flag else None, xv[n:] if self_flag else None)
    np.testing.assert_allclose(dense[n:], cached, rtol=0, atol=1e-13)
    # pair count O(n^2 + nk)
    assert int(mask.sum()) == n * (n + 1) // 2 + n * k + (k if self_flag else 0)
    # candidates never see one another
    off_diag = mask[n:, n:].copy()
    np.fill_diagonal(off_diag, 0)
    assert off_diag.sum() == 0
    # history rows are plain causal attention: check one against an independent numpy softmax
    i = n // 2
    s = (xq[i] @ xk[:i + 1].T) / np.sqrt(d)
    w = np.exp(s - s.max())
    np.testing.assert_allclose(dense[i], (w / w.sum()) @ xv[:i + 1], rtol=0, atol=1e-13)


@pytest.mark.parametrize("self_flag", [False, True])
def test_equals_torch_sdpa_fp64_with_explicit_mask(oracle, self_flag):
    """Library special case: torch SDPA (CPU, fp64) with a boolean mask built here from the
    words of PAPER.md:138, independently of the oracle's mask code."""
    r = rng(10)
    n, k, d = 19, 6, 8
    xq, xk, xv = (r.standard_normal((n + k, d)) for _ in range(3))
    T = n + k
    allow = torch.zeros(T, T, dtype=torch.bool)
    for i in range(T):
        if i < n:
            allow[i, : i + 1] = True
        else:
            allow[i, :n] = True
            allow[i, i] = self_flag
    ref = torch.nn.functional.scaled_dot_product_attention(
        torch.from_numpy(xq)[None, None], torch.from_numpy(xk)[None, None], torch.from_numpy(xv)[None, None],
        attn_mask=allow[None, None])[0, 0].numpy()
    cached = oracle.attn_block(xq[n:], xk[:n], xv[:n], xk[n:] if self_flag else None, xv[n:] if self_flag else None)
    np.testing.assert_allclose(cached, ref[n:], rtol=0, atol=1e-13)
    dense = oracle.full_sequence_attention(xq, xk, xv, n, k, self_flag)
    np.testing.assert_allclose(dense, ref, rtol=0, atol=1e-13)


# ----------------------------------------------------------------------- split-K combine
def test_split_merge_equals_unsplit(oracle):
    r = rng(11)
    C, L, d = 5, 70, 16
    q, K, V = r.standard_normal((C, d)) * 3, r.standard_normal((L, d)), r.standard_normal((L, d))
    full = oracle.attn_block(q, K, V)
    for cuts in ([0, 33, 70], [0, 1, 2, 70], [0, 70, 70], [0, 16, 32, 48, 64, 70]):
        parts = [oracle.attn_partial(q, K, V, a, b) for a, b in zip(cuts[:-1], cuts[1:])]
        m = np.stack([p[0] for p in parts])
        l = np.stack([p[1] for p in parts])
        Ot = np.stack([p[2] for p in parts])
        np.testing.assert_allclose(oracle.combine(m, l, Ot), full, rtol=0, atol=1e-13)


def test_split_merge_with_self_term_as_one_key_range(oracle):
    r = rng(12)
    C, L, d = 4, 20, 8
    q, K, V = r.standard_normal((C, d)), r.standard_normal((L, d)), r.standard_normal((L, d))
    ks, vs = r.standard_normal((C, d)), r.standard_normal((C, d))
    full = oracle.attn_block(q, K, V, ks, vs)
    p0 = oracle.attn_partial(q, K, V, 0, 11)
    p1 = oracle.attn_partial(q, K, V, 11, 20)
    # self range: candidate c against its own key only
    ms, ls, os_ = [], [], []
    for c in range(C):
        m_, l_, o_ = oracle.attn_partial(q[c:c + 1], ks[c:c + 1], vs[c:c + 1], 0, 1)
        ms.append(m_[0]); ls.append(l_[0]); os_.append(o_[0])
    m = np.stack([p0[0], p1[0], np.array(ms)])
    l = np.stack([p0[1], p1[1], np.array(ls)])
    Ot = np.stack([p0[2], p1[2], np.array(os_)])
    np.testing.assert_allclose(oracle.combine(m, l, Ot), full, rtol=0, atol=1e-13)


def test_partial_state_definition_and_empty_ranges(oracle):
    """m = max logit, l = sum exp(s-m), O~ = sum exp(s-m) V -- checked by hand on 2 keys."""
    q = np.array([[2.0, 0.0]])
    K = np.array([[1.0, 0.0], [0.0, 5.0]])
    V = np.array([[10.0, 0.0], [0.0, 20.0]])
    m, l, Ot = oracle.attn_partial(q, K, V, 0, 2, scale=1.0)  # logits 2, 0
    assert m[0] == 2.0
    np.testing.assert_allclose(l[0], 1.0 + np.exp(-2.0), rtol=1e-15)
    np.testing.assert_allclose(Ot[0], [10.0, 20.0 * np.exp(-2.0)], rtol=1e-15)
    m, l, Ot = oracle.attn_partial(q, K, V, 1, 1, scale=1.0)
    assert m[0] == -np.inf and l[0] == 0 and np.all(Ot == 0)
    out = oracle.combine(np.full((2, 1), -np.inf), np.zeros((2, 1)), np.zeros((2, 1, 2)))
    assert np.array_equal(out, np.zeros((1, 2)))


# ----------------------------------------------------------------------- E4M3 codec
def test_e4m3_decode_table_closed_form_and_torch(oracle):
    codes = np.arange(256, dtype=np.uint8)
    dec = oracle.e4m3_decode(codes)
    ref = torch.from_numpy(codes).view(torch.float8_e4m3fn).to(torch.float64).numpy()
    finite = ~np.isnan(ref)
    assert finite.sum() == 254
    assert np.array_equal(dec[finite], ref[finite]) and np.all(np.isnan(dec[~finite]))
    assert dec[0x7E] == 448.0 and dec[0x01] == 2.0 ** -9 and dec[0x08] == 2.0 ** -6 and dec[0x38] == 1.0


def test_e4m3_encode_roundtrip_ties_saturation(oracle):
    codes = np.array([c for c in range(256) if (c & 0x7F) != 0x7F], dtype=np.uint8)
    vals = oracle.e4m3_decode(codes).astype(np.float32)
    enc = oracle.e4m3_encode(vals)
    keep = codes != 0x80  # -0.0 encodes with the sign bit: check separately
    assert np.array_equal(enc[keep], codes[keep])
    assert oracle.e4m3_encode(np.array([-0.0], np.float32))[0] == 0x80
    # constructed midpoints between consecutive positive codes -> even mantissa
    pos = np.arange(0, 0x7E, dtype=np.uint8)
    lo, hi = oracle.e4m3_decode(pos), oracle.e4m3_decode(pos + 1)
    mid = ((lo + hi) / 2).astype(np.float32)  # exact in fp32
    want = np.where(pos % 2 == 0, pos, pos + 1).astype(np.uint8)
    assert np.array_equal(oracle.e4m3_encode(mid), want)
    assert np.array_equal(oracle.e4m3_encode(-mid), want | 0x80)
    # saturation, no NaN/Inf for finite inputs
    assert list(oracle.e4m3_encode(np.array([448, 449, 464, 1e30, -1e30], np.float32))) == [0x7E] * 4 + [0xFE]


def test_e4m3_encode_matches_torch_cast_in_range(oracle):
    r = rng(13)
    x = np.concatenate([r.standard_normal(4000) * s for s in (1e-3, 0.05, 1.0, 30.0, 200.0)]).astype(np.float32)
    x = x[np.abs(x) <= 448.0]
    ref = torch.from_numpy(x).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    assert np.array_equal(oracle.e4m3_encode(x), ref)


def test_bf16_helpers(oracle):
    r = rng(14)
    x = (r.standard_normal(2000) * 10).astype(np.float32)
    bits = oracle.f32_to_bf16_bits(x)
    ref = torch.from_numpy(x).to(torch.bfloat16)
    assert np.array_equal(bits, ref.view(torch.int16).numpy().view(np.uint16))
    assert np.array_equal(oracle.bf16_bits_to_f64(bits), ref.to(torch.float64).numpy())


# ----------------------------------------------------------------------- layout tables and pack
def test_layout_hand_written_cases(oracle):
    lay = oracle.layout([5, 16, 0, 17], H=2, d=64, n_layers=3, dtype=oracle.BF16, align=16, tail_rows=128)
    assert list(lay["row_off"]) == [0, 16, 32, 32, 64]
    assert lay["R"] == 64 and lay["elem_bytes"] == 2 and lay["row_bytes"] == 128
    assert lay["head_stride_bytes"] == 64 * 128 and lay["layer_stride_bytes"] == 2 * 64 * 128
    assert lay["bytes_cache"] == (3 * 2 * 64 + 128) * 128 and lay["bytes_scales"] == 0
    lay8 = oracle.layout([1], H=4, d=128, n_layers=2, dtype=oracle.FP8_E4M3, align=16, tail_rows=128)
    assert list(lay8["row_off"]) == [0, 16] and lay8["bytes_cache"] == (2 * 4 * 16 + 128) * 128
    assert lay8["bytes_scales"] == 2 * 4 * 4
    empty = oracle.layout(np.zeros(0, np.int32), H=1, d=64, n_layers=1, dtype=oracle.BF16)
    assert list(empty["row_off"]) == [0] and empty["R"] == 0


def test_layout_brute_force_properties(oracle):
    r = rng(15)
    for _ in range(20):
        B = int(r.integers(1, 40))
        L = r.integers(0, 300, size=B).astype(np.int32)
        lay = oracle.layout(L, H=3, d=64, n_layers=2, dtype=oracle.BF16)
        ro = lay["row_off"]
        acc = 0
        for b in range(B):
            assert ro[b] == acc and ro[b] % 16 == 0
            acc += -(-int(L[b]) // 16) * 16
        assert ro[B] == acc == lay["R"]
        assert np.all(np.diff(ro) >= L)


def _pool(r, n_layers, S, H, n_max, d):
    x = torch.from_numpy(r.standard_normal((n_layers, S, H, n_max, d)).astype(np.float32)).to(torch.bfloat16)
    return x, x.view(torch.int16).numpy().view(np.uint16)


def test_pack_bf16_is_a_gather_with_zero_padding(oracle):
    r = rng(16)
    n_layers, S, H, n_max, d = 2, 5, 3, 40, 8
    pool_t, pool_bits = _pool(r, n_layers, S, H, n_max, d)
    slot = np.array([3, 0, 4], np.int32)
    L = np.array([7, 40, 0], np.int32)
    cache, scales = oracle.pack(pool_bits, slot, L, oracle.BF16, tail_rows=4)
    assert scales is None
    lay = oracle.layout(L, H, d, n_layers, oracle.BF16, tail_rows=4)
    R, ro = lay["R"], lay["row_off"]
    c = cache.view(np.uint16)[: n_layers * H * R * d].reshape(n_layers, H, R, d)
    want = np.zeros_like(c)
    for l in range(n_layers):
        for b in range(3):
            for h in range(H):
                want[l, h, ro[b]: ro[b] + L[b]] = pool_bits[l, slot[b], h, : L[b]]
    assert np.array_equal(c, want)
    assert np.all(cache.view(np.uint16)[n_layers * H * R * d:] == 0) and cache.size == lay["bytes_cache"]


def test_pack_fp8_scales_and_bytes_against_torch(oracle):
    """scale = amax/448 over the (layer, head)'s valid rows; bytes = RNE-satfinite of x*(448/amax).
    Checked against torch's float8 cast of the same fp32 products."""
    r = rng(17)
    n_layers, S, H, n_max, d = 2, 4, 2, 24, 16
    pool_t, pool_bits = _pool(r, n_layers, S, H, n_max, d)
    slot = np.array([2, 1, 3], np.int32)
    L = np.array([24, 5, 17], np.int32)
    cache, scales = oracle.pack(pool_bits, slot, L, oracle.FP8_E4M3, tail_rows=0)
    lay = oracle.layout(L, H, d, n_layers, oracle.FP8_E4M3, tail_rows=0)
    R, ro = lay["R"], lay["row_off"]
    c = cache.reshape(n_layers, H, R, d)
    pf = pool_t.to(torch.float32)
    for l in range(n_layers):
        for h in range(H):
            amax = max(float(pf[l, slot[b], h, : L[b]].abs().max()) for b in range(3))
            assert scales[l * H + h] == np.float32(amax) / np.float32(448.0)
            mult = np.float32(448.0) / np.float32(amax)
            for b in range(3):
                y = pf[l, slot[b], h, : L[b]] * torch.tensor(mult)
                ref = y.to(torch.float8_e4m3fn).view(torch.uint8).numpy()
                assert np.array_equal(c[l, h, ro[b]: ro[b] + L[b]], ref)
                assert np.all(c[l, h, ro[b] + L[b]: ro[b + 1]] == 0)
            # the extreme element hits +-448 exactly
            assert (np.abs(oracle.e4m3_decode(c[l, h])) == 448.0).any()


def test_pack_fp8_per_user_scales_against_torch_and_single_user_packs(oracle):
    """FP8_E4M3_USER (reading Q18): one scale per (layer, USER, head), amax over that user's valid
    rows only.  Pinned (i) against torch's float8 cast of the same fp32 products and (ii) against the already
    pinned per-(layer, head) pack of each user ALONE (a batch of one has exactly that user's amax)."""
    r = rng(18)
    n_layers, S, H, n_max, d = 2, 4, 2, 24, 16
    pool_t, pool_bits = _pool(r, n_layers, S, H, n_max, d)
    slot = np.array([2, 1, 3, 0], np.int32)
    L = np.array([24, 5, 0, 17], np.int32)
    B = len(L)
    cache, scales = oracle.pack(pool_bits, slot, L, oracle.FP8_E4M3_USER, tail_rows=0)
    lay = oracle.layout(L, H, d, n_layers, oracle.FP8_E4M3_USER, tail_rows=0)
    assert lay["bytes_scales"] == n_layers * B * H * 4 and scales.shape == (n_layers * B * H,)
    R, ro = lay["R"], lay["row_off"]
    c = cache.reshape(n_layers, H, R, d)
    sc = scales.reshape(n_layers, B, H)
    pf = pool_t.to(torch.float32)
    for b in range(B):
        alone, s_alone = oracle.pack(pool_bits, slot[b:b + 1], L[b:b + 1], oracle.FP8_E4M3, tail_rows=0)
        Rb = oracle.layout(L[b:b + 1], H, d, n_layers, oracle.FP8_E4M3, tail_rows=0)["R"]
        alone = alone.reshape(n_layers, H, Rb, d)
        for l in range(n_layers):
            for h in range(H):
                assert sc[l, b, h] == s_alone[l * H + h]
                assert np.array_equal(c[l, h, ro[b]: ro[b] + L[b]], alone[l, h, : L[b]])
                if L[b] == 0:
                    assert sc[l, b, h] == 1.0
                    continue
                amax = float(pf[l, slot[b], h, : L[b]].abs().max())
                assert sc[l, b, h] == np.float32(amax) / np.float32(448.0)
                y = pf[l, slot[b], h, : L[b]] * torch.tensor(np.float32(448.0) / np.float32(amax))
                assert np.array_equal(c[l, h, ro[b]: ro[b] + L[b]], y.to(torch.float8_e4m3fn).view(torch.uint8).numpy())
    # the whole-batch driver indexes the scales per user: equal to per-block calls on the dequantised values
    C = np.array([3, 2, 4, 1])
    co = np.concatenate([[0], np.cumsum(C)]).astype(np.int32)
    q = r.standard_normal((n_layers, co[-1], H, d)).astype(np.float32)
    vc, vs = oracle.pack(pool_bits[:, ::-1].copy(), slot, L, oracle.FP8_E4M3_USER, tail_rows=0)
    out = oracle.cross_attn_packed(q, oracle.F32, cache, vc, oracle.FP8_E4M3_USER, L, co, H, d, n_layers, scales, vs)
    vcr, vsr = vc.reshape(n_layers, H, R, d), vs.reshape(n_layers, B, H)
    for l in range(n_layers):
        for b in range(B):
            for h in range(H):
                K = oracle.e4m3_decode(c[l, h, ro[b]: ro[b] + L[b]]) * float(sc[l, b, h])
                V = oracle.e4m3_decode(vcr[l, h, ro[b]: ro[b] + L[b]]) * float(vsr[l, b, h])
                want = oracle.attn_block(q[l, co[b]:co[b + 1], h].astype(np.float64), K, V)
                np.testing.assert_allclose(out[l, co[b]:co[b + 1], h], want, rtol=0, atol=1e-13)


def test_pack_fp8_zero_head_has_unit_scale(oracle):
    pool = np.zeros((1, 1, 1, 4, 8), np.uint16)
    cache, scales = oracle.pack(pool, [0], [4], oracle.FP8_E4M3, tail_rows=0)
    assert scales[0] == 1.0 and np.all(cache == 0)


# ----------------------------------------------------------------------- whole-batch driver
def test_packed_batch_equals_blockwise(oracle):
    """upro_cross_attn_packed is only indexing + upro_attn_block: check it against per-block
    calls on tensors sliced here with numpy, bf16 and fp8 caches, with and without self."""
    r = rng(18)
    n_layers, H, d = 2, 3, 16
    L = np.array([9, 0, 33], np.int32)
    Cn = np.array([4, 2, 0], np.int32)
    B = 3
    co = np.concatenate([[0], np.cumsum(Cn)]).astype(np.int32)
    tq = int(co[-1])
    n_max = 40
    _, pk = _pool(r, n_layers, B, H, n_max, d)
    _, pv = _pool(r, n_layers, B, H, n_max, d)
    slot = np.array([1, 2, 0], np.int32)
    mk = lambda: torch.from_numpy(r.standard_normal((n_layers, tq, H, d)).astype(np.float32)).to(
        torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    q, ks, vs = mk(), mk(), mk()
    for dt in (oracle.BF16, oracle.FP8_E4M3):
        kc, ksc = oracle.pack(pk, slot, L, dt)
        vc, vsc = oracle.pack(pv, slot, L, dt)
        lay = oracle.layout(L, H, d, n_layers, dt)
        R, ro = lay["R"], lay["row_off"]
        for self_on in (False, True):
            out = oracle.cross_attn_packed(q, oracle.BF16, kc, vc, dt, L, co, H, d, n_layers, ksc, vsc,
                                           ks if self_on else None, vs if self_on else None)
            for l in range(n_layers):
                for b in range(B):
                    for h in range(H):
                        if dt == oracle.BF16:
                            Kd = oracle.bf16_bits_to_f64(kc.view(np.uint16)[: n_layers * H * R * d]).reshape(
                                n_layers, H, R, d)[l, h, ro[b]: ro[b] + L[b]]
                            Vd = oracle.bf16_bits_to_f64(vc.view(np.uint16)[: n_layers * H * R * d]).reshape(
                                n_layers, H, R, d)[l, h, ro[b]: ro[b] + L[b]]
                        else:
                            Kd = oracle.e4m3_decode(kc[: n_layers * H * R * d]).reshape(
                                n_layers, H, R, d)[l, h, ro[b]: ro[b] + L[b]] * float(ksc[l * H + h])
                            Vd = oracle.e4m3_decode(vc[: n_layers * H * R * d]).reshape(
                                n_layers, H, R, d)[l, h, ro[b]: ro[b] + L[b]] * float(vsc[l * H + h])
                        sl = slice(co[b], co[b + 1])
                        qd = oracle.bf16_bits_to_f64(q[l, sl, h])
                        a = (oracle.bf16_bits_to_f64(ks[l, sl, h]), oracle.bf16_bits_to_f64(vs[l, sl, h])) \
                            if self_on else (None, None)
                        if Cn[b] == 0:
                            continue
                        want = oracle.attn_block(qd, Kd, Vd, *a)
                        assert np.array_equal(out[l, sl, h], want)


# ----------------------------------------------------------------------- fp32 branches, user window, pool view
def test_pack_f32_is_exact_widening_of_the_pool(oracle):
    """UPRO_F32 branch of upro_pack: a gather whose elements are the bf16 pool values widened
    exactly -- compared with numpy's own widening (bits << 16 viewed as float32), zero padding."""
    r = rng(21)
    n_layers, S, H, n_max, d = 2, 4, 2, 40, 8
    _, pool_bits = _pool(r, n_layers, S, H, n_max, d)
    slot = np.array([3, 1, 0], np.int32)
    L = np.array([17, 0, 40], np.int32)
    cache, scales = oracle.pack(pool_bits, slot, L, oracle.F32, tail_rows=3)
    assert scales is None
    lay = oracle.layout(L, H, d, n_layers, oracle.F32, tail_rows=3)
    R, ro = lay["R"], lay["row_off"]
    assert cache.size == lay["bytes_cache"] == (n_layers * H * R + 3) * d * 4
    c = cache.view(np.float32)[: n_layers * H * R * d].reshape(n_layers, H, R, d)
    wide = (pool_bits.astype(np.uint32) << 16).view(np.float32)
    want = np.zeros_like(c)
    for l in range(n_layers):
        for b in range(3):
            for h in range(H):
                want[l, h, ro[b]: ro[b] + L[b]] = wide[l, slot[b], h, : L[b]]
    assert np.array_equal(c.view(np.uint32), want.view(np.uint32))
    assert np.all(cache.view(np.float32)[n_layers * H * R * d:] == 0)


def test_packed_batch_f32_cache_and_f32_queries(oracle):
    """UPRO_F32 branch of load_elem (q, k_self, v_self and the cache all fp32): the whole-batch driver
    equals per-block attn_block calls on arrays sliced and widened here with numpy (config 1's dtypes)."""
    r = rng(22)
    n_layers, H, d = 2, 2, 8
    L = np.array([5, 19, 0], np.int32)
    Cn = np.array([3, 2, 4], np.int32)
    B = 3
    co = np.concatenate([[0], np.cumsum(Cn)]).astype(np.int32)
    tq = int(co[-1])
    _, pk = _pool(r, n_layers, B, H, 24, d)
    _, pv = _pool(r, n_layers, B, H, 24, d)
    slot = np.array([2, 0, 1], np.int32)
    # fp32 queries that are NOT bf16-representable: a bf16 misread of the buffer would show
    q, ks, vs = (r.standard_normal((n_layers, tq, H, d)).astype(np.float32) for _ in range(3))
    kc, _ = oracle.pack(pk, slot, L, oracle.F32)
    vc, _ = oracle.pack(pv, slot, L, oracle.F32)
    lay = oracle.layout(L, H, d, n_layers, oracle.F32)
    R, ro = lay["R"], lay["row_off"]
    Kf = kc.view(np.float32)[: n_layers * H * R * d].reshape(n_layers, H, R, d).astype(np.float64)
    Vf = vc.view(np.float32)[: n_layers * H * R * d].reshape(n_layers, H, R, d).astype(np.float64)
    for self_on in (False, True):
        out = oracle.cross_attn_packed(q, oracle.F32, kc, vc, oracle.F32, L, co, H, d, n_layers,
                                       kself=ks if self_on else None, vself=vs if self_on else None)
        for l in range(n_layers):
            for b in range(B):
                for h in range(H):
                    sl = slice(co[b], co[b + 1])
                    a = (ks[l, sl, h].astype(np.float64), vs[l, sl, h].astype(np.float64)) if self_on else (None, None)
                    want = oracle.attn_block(q[l, sl, h].astype(np.float64), Kf[l, h, ro[b]: ro[b] + L[b]],
                                             Vf[l, h, ro[b]: ro[b] + L[b]], *a)
                    assert np.array_equal(out[l, sl, h], want)


def test_packed_batch_user_window(oracle):
    """users=(lo, hi): rows of users inside the window equal the un-windowed call bit for bit, rows
    outside stay zero; windows tile the batch; an empty window computes nothing."""
    r = rng(23)
    n_layers, H, d = 1, 2, 8
    L = np.array([5, 19, 0, 33, 7], np.int32)
    Cn = np.array([3, 2, 4, 1, 5], np.int32)
    B = 5
    co = np.concatenate([[0], np.cumsum(Cn)]).astype(np.int32)
    tq = int(co[-1])
    _, pk = _pool(r, n_layers, B, H, 40, d)
    _, pv = _pool(r, n_layers, B, H, 40, d)
    slot = np.arange(B, dtype=np.int32)[::-1].copy()
    mk = lambda: torch.from_numpy(r.standard_normal((n_layers, tq, H, d)).astype(np.float32)).to(
        torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    q, ks, vs = mk(), mk(), mk()
    kc, _ = oracle.pack(pk, slot, L, oracle.BF16)
    vc, _ = oracle.pack(pv, slot, L, oracle.BF16)
    full = oracle.cross_attn_packed(q, oracle.BF16, kc, vc, oracle.BF16, L, co, H, d, n_layers, kself=ks, vself=vs)
    assert np.abs(full).min(axis=(0, 2, 3)).max() > 0          # every candidate row is populated
    acc = np.zeros_like(full)
    for lo, hi in ((0, 2), (2, 2), (2, 4), (4, 5)):
        part = oracle.cross_attn_packed(q, oracle.BF16, kc, vc, oracle.BF16, L, co, H, d, n_layers,
                                        kself=ks, vself=vs, users=(lo, hi))
        assert np.array_equal(part[:, co[lo]:co[hi]], full[:, co[lo]:co[hi]])
        assert np.all(part[:, :co[lo]] == 0) and np.all(part[:, co[hi]:] == 0)
        acc += part
    assert np.array_equal(acc, full)


@pytest.mark.parametrize("G", [1, 2, 4])
def test_pool_addressed_batch_equals_pack_then_attend(oracle, G):
    """upro_cross_attn_pool (zero-copy addressing of PAPER.md:202's pool, grouped queries) against
    (i) per-block attn_block calls on pool slices taken here with numpy, and, for G == 1, (ii) the
    packed path: pack (PAPER.md:204's slot copy) then upro_cross_attn_packed -- the copy must not
    change the result."""
    r = rng(24 + G)
    n_layers, H_kv, d = 2, 2, 8
    H_q = H_kv * G
    L = np.array([9, 0, 33, 16], np.int32)
    Cn = np.array([4, 2, 0, 3], np.int32)
    B, S = 4, 6
    co = np.concatenate([[0], np.cumsum(Cn)]).astype(np.int32)
    tq = int(co[-1])
    _, pk = _pool(r, n_layers, S, H_kv, 40, d)
    _, pv = _pool(r, n_layers, S, H_kv, 40, d)
    slot = np.array([5, 2, 0, 3], np.int32)
    mk = lambda: torch.from_numpy(r.standard_normal((n_layers, tq, H_q, d)).astype(np.float32)).to(
        torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    q, ks, vs = mk(), mk(), mk()
    for self_on in (False, True):
        kw = dict(kself=ks, vself=vs) if self_on else {}
        out = oracle.cross_attn_pool(q, oracle.BF16, pk, pv, slot, L, co, H_q, **kw)
        for l in range(n_layers):
            for b in range(B):
                for hq in range(H_q):
                    if Cn[b] == 0:
                        continue
                    sl = slice(co[b], co[b + 1])
                    Kd = oracle.bf16_bits_to_f64(pk[l, slot[b], hq // G, : L[b]])
                    Vd = oracle.bf16_bits_to_f64(pv[l, slot[b], hq // G, : L[b]])
                    a = (oracle.bf16_bits_to_f64(ks[l, sl, hq]), oracle.bf16_bits_to_f64(vs[l, sl, hq])) \
                        if self_on else (None, None)
                    assert np.array_equal(out[l, sl, hq], oracle.attn_block(oracle.bf16_bits_to_f64(q[l, sl, hq]),
                                                                            Kd, Vd, *a))
        if G == 1:
            kc, _ = oracle.pack(pk, slot, L, oracle.BF16)
            vc, _ = oracle.pack(pv, slot, L, oracle.BF16)
            packed = oracle.cross_attn_packed(q, oracle.BF16, kc, vc, oracle.BF16, L, co, H_q, d, n_layers, **kw)
            assert np.array_equal(out, packed)
    with pytest.raises(ValueError):
        oracle.cross_attn_pool(q, oracle.BF16, pk, pv, np.array([5, 2, 0, 6], np.int32), L, co, H_q)  # slot >= S
