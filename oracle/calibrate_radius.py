"""TEST INFRASTRUCTURE — writes the stored per-config radius r^2 (SURVEY.md Q4 / DESIGN.md readings).

BASELINE.json fixes the radius only as "r set for mean out-degree 6" (10 for the stress config).
Reading: once per config, on seeded calibration events (C0/C1: the event itself; C2/C4: the first 16
events; C3 shares C2's), compute the ORACLE's fp32 embeddings, collect every candidate pair's d^2 in
double, take k = round(target * N_cal) and set r^2 = midpoint between the k-th and (k+1)-th smallest,
rounded to fp32.  The constant is stored in paper_2508_07423_b200/config_constants.json and read by
both paths; nothing here touches the CUDA library.

Run:  python -m oracle.calibrate_radius
"""
from __future__ import annotations

import json
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

from oracle import etx_oracle as orc  # noqa: E402
from paper_2508_07423_b200 import synth  # noqa: E402  (input generator only)


def calibrate(name: str) -> dict:
    cfg = synth.CONFIGS[name]
    batch = synth.generate_events(cfg, range(min(cfg.calib_events, cfg.n_events)))
    blob = synth.generate_weights(cfg)
    emb_spec = synth.model_layout(cfg)[0]
    fe, _ = orc.features(batch, synth.NORM_CENTER, synth.NORM_SCALE)
    emb = orc.mlp(fe, emb_spec.dims, blob, emb_spec.offset)
    d2 = np.sort(orc.candidate_d2(batch["event_ptr"], batch["plane"], emb, cfg.max_plane_gap))
    n_cal = len(batch["r"])
    k = int(np.floor(cfg.target_degree * n_cal + 0.5))
    k = min(max(k, 1), len(d2) - 1)
    r2 = np.float32(0.5 * (d2[k - 1] + d2[k]))
    src, _ = orc.build_graph(batch["event_ptr"], batch["plane"], emb, float(r2), cfg.max_plane_gap)
    return {"r2_max": float(r2), "calib_hits": int(n_cal), "calib_candidates": int(len(d2)),
            "calib_edges": int(len(src)), "calib_mean_out_degree": float(len(src)) / n_cal,
            "target_degree": cfg.target_degree, "max_plane_gap": cfg.max_plane_gap}


def main():
    path = os.path.join(os.path.dirname(os.path.abspath(synth.__file__)), "config_constants.json")
    out = {}
    if os.path.exists(path):                      # keep what other calibration scripts stored (oracle/calibrate_int8.py)
        with open(path) as f:
            out = json.load(f)
    for name in ("c0", "c1", "c2", "c4"):
        out.setdefault(name, {}).update(calibrate(name))
    with open(path, "w") as f:
        json.dump(out, f, indent=1, sort_keys=True)
        f.write("\n")
    print(json.dumps(out, indent=1, sort_keys=True))


if __name__ == "__main__":
    main()
