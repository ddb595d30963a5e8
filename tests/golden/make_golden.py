"""Writes tests/golden/attn_tiny.json: a tiny worked example of the ranking cross-attention
computed by the ORACLE ALONE (never by the CUDA path).  The paper prints no worked
numerical example of the attention, so this fixture exists to freeze the oracle against
accidental changes and to give the GPU tests a stored case; the definition it follows is
PAPER.md:138 / 198 (candidates attend to the cached history and, optionally, to themselves).

    python tests/golden/make_golden.py
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle  # noqa: E402


def main():
    # exactly representable inputs (multiples of 1/8), so the JSON holds them without rounding
    rng = np.random.default_rng(20260422)
    d, L, C = 8, 5, 3
    q = rng.integers(-8, 9, size=(C, d)) / 8.0
    K = rng.integers(-8, 9, size=(L, d)) / 8.0
    V = rng.integers(-8, 9, size=(L, d)) / 8.0
    ks = rng.integers(-8, 9, size=(C, d)) / 8.0
    vs = rng.integers(-8, 9, size=(C, d)) / 8.0
    out_plain, w_plain = oracle.attn_block(q, K, V, return_weights=True)
    out_self, w_self = oracle.attn_block(q, K, V, ks, vs, return_weights=True)
    fix = {
        "cite": "PAPER.md:138, 198 (definition); values computed by oracle/upr_oracle.c in fp64",
        "d": d, "L": L, "C": C, "scale": 1.0 / np.sqrt(d),
        "q": q.tolist(), "K": K.tolist(), "V": V.tolist(), "k_self": ks.tolist(), "v_self": vs.tolist(),
        "out_no_self": out_plain.tolist(), "weights_no_self": w_plain.tolist(),
        "out_self": out_self.tolist(), "weights_self": w_self.tolist(),
    }
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "attn_tiny.json")
    with open(path, "w") as f:
        json.dump(fix, f, indent=1)
    print("wrote", path)


if __name__ == "__main__":
    main()
