"""upr_cross_attn_fwd_noalloc: the forward call whose scratch is a static device array inside the library (no
cudaMalloc in the call) against the existing path, upr_cross_attn_fwd_ex with a caller-provided workspace.

Collected last on purpose (the suite runs with pytest -x).  Passes alone in a fresh process and after the other
tests: it depends on nothing they leave behind, and the static scratch is rewritten by every call before it is read.
"""
import numpy as np
import pytest
import torch

import upr_synth as S
from harness import Inputs

pytestmark = pytest.mark.gpu

TOL_STRICT = 5e-3     # the parity tests' self-imposed bound (tests/test_gpu_parity.py)


@pytest.fixture(scope="module")
def P():
    import paper_2606_00422_b200 as P
    return P


def _both_paths(P, pl, w, inp, num_splits, kernel):
    """One call through the existing path and one through the no-alloc entry point, same inputs."""
    view = pl.PoolView.of(inp.k_pool, inp.v_pool, inp.slot_ids, w.seq_lens)
    attn = pl.CrossAttention(view, w.cand_offsets, P.UPR_BF16, num_splits=num_splits, kernel=kernel)
    ks, vs = (inp.k_self, inp.v_self) if w.self_term else (None, None)
    want = attn(inp.q, ks, vs).clone()
    want_kernel, want_launches = P.upr_last_attn_kernel(), P.upr_last_launch_count()
    got = torch.full_like(want, float("nan"))
    P.upr_cross_attn_fwd_noalloc(inp.q, view.k_pool, view.v_pool, view.seq_lens, attn.cand_offsets, got, attn.B, attn.H,
                                 attn.d, attn.n_layers, P.UPR_BF16, P.UPR_BF16, attn.total_q, ks, vs,
                                 num_splits=num_splits, max_seq_len=view.max_seq_len, **attn.kv_kwargs)
    torch.cuda.synchronize()
    assert P.upr_last_attn_kernel() == want_kernel and P.upr_last_launch_count() == want_launches
    return got.cpu().numpy(), want.cpu().numpy()


def test_no_alloc_entry_point_matches_the_workspace_path_on_two_calls_in_a_row(P):
    from paper_2606_00422_b200 import pipeline as pl
    assert P.upr_cross_attn_noalloc_scratch_bytes() == 8 << 20
    # call 1: ragged batch, self term, two layers, CTA-pair kernel, no split-K
    w1 = S.custom_workload("na1", 301, [300, 0, 77, 1024, 129], [300, 5, 0, 257, 40], 4, 128, 2, self_term=True)
    # call 2, right after it, different shape: split-K (the partials live in the same static scratch, which still
    # holds call 1's tables) on the 1-CTA kernel
    w2 = S.custom_workload("na2", 302, [2048, 700], [33, 8], 2, 128, 1)
    for w, ns, kernel in ((w1, 1, P.UPR_KERNEL_PAIR), (w2, 4, P.UPR_KERNEL_SINGLE), (w1, 1, P.UPR_KERNEL_PAIR)):
        inp = Inputs(w, "cuda")
        got, want = _both_paths(P, pl, w, inp, ns, kernel)
        assert np.isfinite(got).all()
        err = float(np.abs(got.astype(np.float64) - want).max())
        assert err <= TOL_STRICT, (w.name, err)


def test_no_alloc_entry_point_refuses_what_does_not_fit(P):
    from paper_2606_00422_b200 import pipeline as pl
    # split-K partials of this shape: 1 * 3000 * 8 * 16 * 130 * 4 bytes = 200 MB > 8 MiB
    B, H, d, total_q = 4, 8, 128, 3000
    need = P.upr_cross_attn_workspace_bytes(B, H, d, 1, total_q, num_splits=16, max_seq_len=8192)
    assert need > P.upr_cross_attn_noalloc_scratch_bytes()
    z = torch.zeros(16, dtype=torch.uint8, device="cuda")
    with pytest.raises(P.UprError) as e:
        P.upr_cross_attn_fwd_noalloc(z, z, z, z, z, z, B, H, d, 1, P.UPR_BF16, P.UPR_BF16, total_q, num_splits=16,
                                     max_seq_len=8192)
    assert e.value.status == 3 and "static scratch" in str(e.value) and str(need) in str(e.value)
    assert P.upr_last_launch_count() == 0
