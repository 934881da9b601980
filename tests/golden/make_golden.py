"""Writes tests/golden/c0_oracle.txt from the ORACLE only (never from the CUDA path).

A regression guard on the oracle itself: a later change to its arithmetic must be deliberate (and, per
DESIGN.md, justified by a passage of the thesis in the commit message) because this file changes.
Run:  python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import etx_oracle as orc  # noqa: E402
from paper_2508_07423_b200 import synth  # noqa: E402


def compute():
    cfg = synth.CONFIGS["c0"]
    b = synth.generate_events(cfg)
    blob = synth.generate_weights(cfg)
    lo = {s.name: (s.dims, s.offset) for s in synth.model_layout(cfg)}
    out = orc.run_path(b, blob, lo, cfg.gnn_hidden, cfg.n_iter, synth.r2_max(cfg), cfg.max_plane_gap,
                       synth.NORM_CENTER, synth.NORM_SCALE)
    return {"n_hits": len(b["r"]), "n_edges": len(out["src"]),
            "edge_checksum": int((out["src"].astype(np.int64) * 7919 + out["dst"]).sum()),
            "first_scores": [float(x) for x in out["scores"][:8]],
            "score_sum": float(out["scores"].astype(np.float64).sum())}


if __name__ == "__main__":
    g = compute()
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "c0_oracle.txt"), "w") as f:
        f.write("# written by tests/golden/make_golden.py from oracle/ only (config C0)\n")
        for k, v in g.items():
            f.write(f"{k} = {v!r}\n")
    print(g)
