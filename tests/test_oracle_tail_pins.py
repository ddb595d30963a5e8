"""Pins for the oracle's decode-layer tail and consumer: the linear
layer, the per-action MLP heads with their utility (PAPER.md:146-152 Eq. 4, :321) and the
per-user top-K.  None of these re-types the oracle's formula: library routines (numpy matmul,
torch.nn.functional), hand-computed values, invariants and brute force.  -m "not gpu"."""
import numpy as np
import torch


def rng(seed):
    return np.random.default_rng(seed)


# ----------------------------------------------------------------------------- linear
def test_linear_equals_library_matmul(oracle):
    r = rng(0)
    for (M, N, K) in [(1, 1, 1), (5, 3, 7), (33, 17, 64), (4, 130, 9)]:
        x, w, b = r.standard_normal((M, K)), r.standard_normal((N, K)), r.standard_normal(N)
        np.testing.assert_allclose(oracle.linear(x, w), x @ w.T, rtol=0, atol=1e-12)
        np.testing.assert_allclose(oracle.linear(x, w, b), x @ w.T + b, rtol=0, atol=1e-12)


def test_linear_hand_case_catches_a_transposed_operand(oracle):
    # W = [[1,2],[3,4],[5,6]] is [N=3, K=2]: y_n = <x, W[n]>; with x = (1, 10): (21, 43, 65)
    y = oracle.linear(np.array([[1.0, 10.0]]), np.array([[1.0, 2.0], [3.0, 4.0], [5.0, 6.0]]),
                      np.array([0.5, 0.0, -1.0]))
    np.testing.assert_array_equal(y, [[21.5, 43.0, 64.0]])


def test_linear_activations_against_torch(oracle):
    r = rng(1)
    x, w, b = r.standard_normal((9, 5)), r.standard_normal((4, 5)), r.standard_normal(4)
    pre = torch.from_numpy(x @ w.T + b)
    np.testing.assert_allclose(oracle.linear(x, w, b, act=oracle.ACT_SILU),
                               torch.nn.functional.silu(pre).numpy(), rtol=0, atol=1e-13)
    np.testing.assert_allclose(oracle.linear(x, w, b, act=oracle.ACT_RELU),
                               torch.relu(pre).numpy(), rtol=0, atol=1e-13)
    # closed forms: silu(0) = 0, silu(t) -> t for large t, silu(-t) -> 0
    y = oracle.linear(np.array([[0.0], [40.0], [-40.0]]), np.array([[1.0]]), act=oracle.ACT_SILU)
    np.testing.assert_allclose(y[:, 0], [0.0, 40.0, 0.0], rtol=0, atol=1e-15)


def test_linear_is_linear_and_composes(oracle):
    """Invariants: additivity in x; two layers without activation == one layer with the product."""
    r = rng(2)
    x1, x2 = r.standard_normal((6, 8)), r.standard_normal((6, 8))
    w, w2 = r.standard_normal((5, 8)), r.standard_normal((3, 5))
    np.testing.assert_allclose(oracle.linear(x1 + x2, w), oracle.linear(x1, w) + oracle.linear(x2, w),
                               rtol=0, atol=1e-13)
    np.testing.assert_allclose(oracle.linear(oracle.linear(x1, w), w2), oracle.linear(x1, w2 @ w),
                               rtol=0, atol=1e-12)


# ----------------------------------------------------------------------------- action heads
def _heads(r, C, Dh, D):
    return (r.standard_normal((C, Dh, D)) / np.sqrt(D), r.standard_normal((C, Dh)) * 0.1,
            r.standard_normal((C, Dh)) / np.sqrt(Dh), r.standard_normal(C) * 0.1, r.uniform(0.1, 2.0, C))


def test_action_utility_against_torch_modules(oracle):
    """Each head is Linear -> SiLU -> Linear(1) -> sigmoid; utility = sum_c w_c p_c (Eq. 4's heads and
    weights).  torch.nn.functional supplies every step."""
    r = rng(3)
    M, D, C, Dh = 11, 16, 3, 8
    z = r.standard_normal((M, D))
    w1, b1, w2, b2, wc = _heads(r, C, Dh, D)
    probs, util = oracle.action_utility(z, w1, b1, w2, b2, wc)
    F = torch.nn.functional
    zt = torch.from_numpy(z)
    want = torch.stack([torch.sigmoid(F.linear(F.silu(F.linear(zt, torch.from_numpy(w1[c]), torch.from_numpy(b1[c]))),
                                               torch.from_numpy(w2[c:c + 1]), torch.from_numpy(b2[c:c + 1])))[:, 0]
                        for c in range(C)], dim=1).numpy()
    np.testing.assert_allclose(probs, want, rtol=0, atol=1e-13)
    np.testing.assert_allclose(util, want @ wc, rtol=0, atol=1e-13)


def test_action_utility_closed_forms(oracle):
    # zero weights: logit = b2 -> p = sigmoid(b2); b2 = 0 -> 1/2 each -> utility = sum(w)/2
    M, D, C, Dh = 4, 6, 3, 5
    z = rng(4).standard_normal((M, D))
    zero = np.zeros
    probs, util = oracle.action_utility(z, zero((C, Dh, D)), zero((C, Dh)), zero((C, Dh)), zero(C),
                                        np.array([1.0, 2.0, 4.0]))
    np.testing.assert_array_equal(probs, 0.5)
    np.testing.assert_allclose(util, 3.5, rtol=0, atol=1e-15)
    probs, _ = oracle.action_utility(z, zero((C, Dh, D)), zero((C, Dh)), zero((C, Dh)), np.array([np.log(3.0), 0, -np.log(3.0)]),
                                     np.ones(C))
    np.testing.assert_allclose(probs[0], [0.75, 0.5, 0.25], rtol=0, atol=1e-15)


def test_action_utility_rows_and_heads_are_independent(oracle):
    """A candidate's probabilities do not depend on the batch; head c uses only its own
    parameters (PAPER.md:146 'a dedicated MLP head')."""
    r = rng(5)
    M, D, C, Dh = 7, 8, 4, 6
    z = r.standard_normal((M, D))
    w1, b1, w2, b2, wc = _heads(r, C, Dh, D)
    probs, util = oracle.action_utility(z, w1, b1, w2, b2, wc)
    perm = r.permutation(M)
    p2, u2 = oracle.action_utility(z[perm], w1, b1, w2, b2, wc)
    np.testing.assert_array_equal(p2, probs[perm])
    np.testing.assert_array_equal(u2, util[perm])
    w1b = w1.copy()
    w1b[2] += 1.0                      # perturb head 2 only
    p3, _ = oracle.action_utility(z, w1b, b1, w2, b2, wc)
    np.testing.assert_array_equal(p3[:, [0, 1, 3]], probs[:, [0, 1, 3]])
    assert np.abs(p3[:, 2] - probs[:, 2]).max() > 1e-6
    # head c alone == the same head through the linear oracle
    hid = oracle.linear(z, w1[1], b1[1], act=oracle.ACT_SILU)
    np.testing.assert_allclose(probs[:, 1], 1 / (1 + np.exp(-(hid @ w2[1] + b2[1]))), rtol=0, atol=1e-13)


# ----------------------------------------------------------------------------- top-K
def test_topk_hand_case_with_ties(oracle):
    #          user 0: 4 cands          user 1: none   user 2: 2 cands
    util = np.array([0.5, 0.9, 0.9, 0.1, 0.3, 0.7], dtype=np.float32)
    idx, cnt = oracle.topk_per_user(util, [0, 4, 4, 6], 3)
    np.testing.assert_array_equal(cnt, [3, 0, 2])
    np.testing.assert_array_equal(idx, [[1, 2, 0], [-1, -1, -1], [5, 4, -1]])   # tie 0.9/0.9 -> lower index first


def test_topk_brute_force_against_stable_argsort(oracle):
    r = rng(6)
    for trial in range(5):
        B = int(r.integers(1, 9))
        counts = r.integers(0, 40, size=B)
        co = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
        util = r.integers(0, 6, size=co[-1]).astype(np.float32) / 4    # many ties
        K = int(r.integers(1, 12))
        idx, cnt = oracle.topk_per_user(util, co, K)
        for b in range(B):
            seg = util[co[b]:co[b + 1]]
            order = np.argsort(-seg, kind="stable")[:K] + co[b]       # descending, ties by index
            assert cnt[b] == min(K, len(seg))
            np.testing.assert_array_equal(idx[b, :cnt[b]], order)
            assert np.all(idx[b, cnt[b]:] == -1)


# ----------------------------------------------------------------------------- layer norm
def test_layernorm_against_torch_and_closed_forms(oracle):
    r = rng(7)
    x, g, b = r.standard_normal((6, 32)) * 3 + 1, r.standard_normal(32), r.standard_normal(32)
    want = torch.nn.functional.layer_norm(torch.from_numpy(x), (32,), torch.from_numpy(g), torch.from_numpy(b), 1e-5)
    np.testing.assert_allclose(oracle.layernorm(x, g, b), want.numpy(), rtol=0, atol=1e-12)
    # gamma = 1, beta = 0: zero mean, unit variance (up to eps); a shift and a positive scale of x change nothing
    y = oracle.layernorm(x, np.ones(32), np.zeros(32), eps=0.0)
    np.testing.assert_allclose(y.mean(axis=1), 0.0, atol=1e-14)
    np.testing.assert_allclose((y ** 2).mean(axis=1), 1.0, atol=1e-13)
    np.testing.assert_allclose(oracle.layernorm(5.0 * x + 7.0, np.ones(32), np.zeros(32), eps=0.0), y, atol=1e-12)
    # hand case: x = (1, 3): mean 2, var 1 -> (-1, 1) * gamma + beta
    np.testing.assert_allclose(oracle.layernorm(np.array([[1.0, 3.0]]), np.array([2.0, 3.0]), np.array([0.5, -0.5]), eps=0.0),
                               [[-1.5, 2.5]], atol=1e-15)


# ----------------------------------------------------------------------------- FP8 linear
def test_linear_fp8_against_torch_float8_and_the_exact_case(oracle):
    r = rng(8)
    M, N, K = 7, 5, 32
    x = r.standard_normal((M, K)).astype(np.float32)
    w = r.standard_normal((N, K)).astype(np.float32)
    xs, ws = np.float32(np.abs(x).max() / 448.0), np.float32(np.abs(w).max() / 448.0)
    w8 = torch.from_numpy(w * (np.float32(1.0) / ws)).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    got = oracle.linear_fp8(x, float(xs), w8, float(ws))
    # torch's float8 cast as the library routine for both operands
    xq = torch.from_numpy(x * (np.float32(1.0) / xs)).to(torch.float8_e4m3fn).to(torch.float64).numpy()
    wq = torch.from_numpy(w8).view(torch.float8_e4m3fn).to(torch.float64).numpy()
    np.testing.assert_allclose(got, (xq @ wq.T) * float(xs) * float(ws), rtol=0, atol=1e-12)
    # quantisation error is what FP8 costs: ~2^-4 relative per operand, averaged over K
    assert np.abs(got - x.astype(np.float64) @ w.astype(np.float64).T).max() < 0.6
    # operands that are exactly representable with scale 1: identical to the plain linear layer
    xi = r.integers(-8, 9, size=(M, K)).astype(np.float32)
    wi = r.integers(-8, 9, size=(N, K)).astype(np.float32)
    wi8 = oracle.e4m3_encode(wi)
    np.testing.assert_array_equal(oracle.linear_fp8(xi, 1.0, wi8, 1.0), oracle.linear(xi, wi))
    # scales factor out: y(x, 2 x_scale) with x doubled == 2 y
    np.testing.assert_allclose(oracle.linear_fp8(2 * xi, 2.0, wi8, 1.0), 2 * oracle.linear(xi, wi), rtol=0, atol=1e-12)


def test_linear_fp8q_is_the_plain_layer_on_decoded_bytes(oracle):
    """Activations that arrive as E4M3 bytes: pinned to torch's float8 decode + a float64 matmul (library routines), to
    upro_linear_fp8 on the decoded values (quantising a representable value is the identity), and to the exact
    integer case."""
    r = rng(9)
    M, N, K = 6, 5, 64
    x8 = r.integers(0, 256, size=(M, K)).astype(np.uint8)
    w8 = r.integers(0, 256, size=(N, K)).astype(np.uint8)
    x8[(x8 & 0x7F) == 0x7F] = 0x38          # no NaN codes
    w8[(w8 & 0x7F) == 0x7F] = 0xB8
    b = r.standard_normal(N)
    xs, ws = 0.25, 0.03125
    got = oracle.linear_fp8q(x8, xs, w8, ws, b, act=oracle.ACT_RELU)
    xd = torch.from_numpy(x8).view(torch.float8_e4m3fn).to(torch.float64).numpy()
    wd = torch.from_numpy(w8).view(torch.float8_e4m3fn).to(torch.float64).numpy()
    np.testing.assert_allclose(got, np.maximum((xd @ wd.T) * xs * ws + b, 0.0), rtol=0, atol=1e-9)
    # the in-kernel-quantising layer fed the decoded values (scale 1: x * 1.0f is exact, encode(decode(b)) == b)
    np.testing.assert_array_equal(oracle.linear_fp8q(x8, 1.0, w8, ws, b), oracle.linear_fp8(xd.astype(np.float32), 1.0, w8, ws, b))
    xi = r.integers(-8, 9, size=(M, K)).astype(np.float32)
    wi = r.integers(-8, 9, size=(N, K)).astype(np.float32)
    np.testing.assert_array_equal(oracle.linear_fp8q(oracle.e4m3_encode(xi), 1.0, oracle.e4m3_encode(wi), 1.0), oracle.linear(xi, wi))
