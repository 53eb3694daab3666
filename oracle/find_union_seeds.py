"""Rejection-sample the try seeds of BASELINE.json configs 2 and 3: for each (T, u)
find the first seed whose gate-driven active-expert union has exactly min(u, T*k) experts.  The realised union is
the ONLY acceptance criterion: near-tie tokens are not filtered out here -- the parity tests
classify them per token (margin <= 1e-5) and report them; the recorded min_margin is information only.

Calls ONLY the oracle (oracle/eldr_oracle.c) and the seeded generators; writes
paper_2607_00466_b200/union_seeds.json (an input recipe, not an expected value).
Run from the repo root:  python oracle/find_union_seeds.py
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from oracle import oracle  # noqa: E402
from paper_2607_00466_b200 import synth  # noqa: E402

CASES = [(64, u) for u in (16, 32, 64, 96, 128)] + [(T, 32) for T in (1, 8, 32, 128, 256)]


def main():
    shape = synth.SHAPE_QWEN
    gate_w = synth.make_gate_w(shape, synth.WEIGHT_SEED, 0)
    out = {}
    for T, u in CASES:
        want = min(u, T * shape.top_k)
        for seed in range(1000, 3000):
            x, bias = synth.union_case(shape, T, u, seed)
            r = oracle.gate_topk(shape, x, gate_w, bias)
            realised = len(np.unique(r["ids"]))
            if realised == want:
                out["T%d_u%d" % (T, u)] = {"seed": seed, "union": realised, "tries": seed - 999,
                                           "min_margin": float(r["margin"].min())}
                print(T, u, out["T%d_u%d" % (T, u)])
                break
        else:
            raise SystemExit("no seed for T=%d u=%d" % (T, u))
    path = os.path.join(ROOT, "paper_2607_00466_b200", "union_seeds.json")
    with open(path, "w") as f:
        json.dump(out, f, indent=1, sort_keys=True)
    print("wrote", path)


if __name__ == "__main__":
    main()
