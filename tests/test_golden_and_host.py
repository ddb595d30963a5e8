"""CPU-only checks: the stored oracle fixture against an independent numpy evaluation of the
definition, the host-side layout call of the C-ABI library, its exported symbols, and the
multi-rank aggregation used by bench.py (world size 2, gloo)."""
import ctypes
import json
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
GOLD = os.path.join(ROOT, "tests", "golden", "attn_tiny.json")


def _softmax_attention(q, K, V, ks=None, vs=None):
    """The definition in plain numpy fp64: logits, softmax, weighted sum."""
    d = q.shape[1]
    out = np.zeros_like(q)
    for c in range(q.shape[0]):
        s = K @ q[c] / np.sqrt(d)
        vals = V
        if ks is not None:
            s = np.append(s, ks[c] @ q[c] / np.sqrt(d))
            vals = np.vstack([V, vs[c]])
        w = np.exp(s - s.max())
        out[c] = (w / w.sum()) @ vals
    return out


def test_golden_fixture_matches_oracle_and_numpy(oracle):
    g = json.load(open(GOLD))
    q, K, V = np.array(g["q"]), np.array(g["K"]), np.array(g["V"])
    ks, vs = np.array(g["k_self"]), np.array(g["v_self"])
    # the oracle still reproduces what it wrote
    assert np.allclose(oracle.attn_block(q, K, V), np.array(g["out_no_self"]), atol=1e-15)
    assert np.allclose(oracle.attn_block(q, K, V, ks, vs), np.array(g["out_self"]), atol=1e-15)
    # and the stored values are the definition evaluated independently
    assert np.allclose(_softmax_attention(q, K, V), np.array(g["out_no_self"]), atol=1e-13)
    assert np.allclose(_softmax_attention(q, K, V, ks, vs), np.array(g["out_self"]), atol=1e-13)
    assert np.allclose(np.array(g["weights_self"]).sum(axis=1), 1.0, atol=1e-14)
    # the self weight is the last column; without the self term it is zero
    assert np.all(np.array(g["weights_no_self"])[:, -1] == 0.0)


def test_library_loads_and_exports_every_declared_symbol():
    import paper_2606_00422_b200 as P
    lib = ctypes.CDLL(P.lib_path())
    header = open(os.path.join(ROOT, "include", "upr.h")).read()
    for name in P.EXPORTED_SYMBOLS:
        assert name + "(" in header, f"{name} not declared in upr.h"
        assert getattr(lib, name) is not None
    assert P.upr_version().startswith("upr")


def test_host_layout_call_matches_oracle_without_a_gpu(oracle):
    import paper_2606_00422_b200 as P
    rng = np.random.default_rng(5)
    for dt, odt in ((P.UPR_BF16, oracle.BF16), (P.UPR_FP8_E4M3, oracle.FP8_E4M3), (P.UPR_F32, oracle.F32)):
        L = rng.integers(0, 5000, size=37).astype(np.int32)
        lay, ro = P.upr_kv_cache_layout(L, 16, 64, 2, dt)
        o = oracle.layout(L, 16, 64, 2, odt, align=P.UPR_ROW_ALIGN, tail_rows=P.UPR_TAIL_ROWS)
        assert np.array_equal(ro, o["row_off"]) and lay.R == o["R"] and lay.bytes_cache == o["bytes_cache"]
        assert lay.bytes_scales == o["bytes_scales"]
    with pytest.raises(P.UprError):
        P.upr_kv_cache_layout([1], 2, 80, 1, P.UPR_BF16)          # unsupported head dim


def test_workspace_and_split_policy_are_host_only():
    import paper_2606_00422_b200 as P
    # plenty of items: no split, workspace = scheduler counter block + work-list tables (3 x (B+1) int32,
    # rounded up to 256 bytes)
    def tables(B):
        return (3 * (B + 1) * 4 + 255) // 256 * 256
    assert P.upr_cross_attn_num_splits(256, 8, 128, 4, 131072, 0, 2048) == 1
    assert P.upr_cross_attn_workspace_bytes(256, 8, 128, 4, 131072, 0, 2048) == 256 + tables(256)
    # one user, few candidates, long history: the heuristic splits the history
    ns = P.upr_cross_attn_num_splits(1, 2, 128, 1, 16, 0, 8192)
    assert ns > 1
    need = P.upr_cross_attn_workspace_bytes(1, 2, 128, 1, 16, 0, 8192)
    assert need == 256 + tables(1) + 16 * 2 * ns * (128 + 2) * 4
    assert P.upr_cross_attn_num_splits(1, 2, 128, 1, 16, 3, 8192) == 3   # explicit request wins


_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo", rank=int(os.environ["RANK"]), world_size=2,
                        init_method="tcp://127.0.0.1:{port}")
rank = dist.get_rank()
# rank r reports (10 + 5 r) ms and (100 + r) units: the job took the slower rank's time and did the sum
ms, units = bench.aggregate_over_ranks(10.0 + 5.0 * rank, 100 + rank, dist)
assert ms == 15.0 and units == 201, (ms, units)
w0, w1 = bench.rank_workload(2, 0), bench.rank_workload(2, 1)
assert w0.seed != w1.seed and w0.B == w1.B       # same config, rank-specific batch: weak scaling
dist.destroy_process_group()
print("ok", rank)
"""


def test_multi_rank_aggregation_world_size_2_gloo(tmp_path):
    """N > 1 path of bench.py: users shard by rank with no data-path collective; only the timing
    (max over ranks) and the unit count (sum over ranks) are reduced."""
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT, port=29500 + os.getpid() % 1000))
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=240)[0] for p in procs]
    for p, o in zip(procs, outs):
        assert p.returncode == 0, o
