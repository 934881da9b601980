"""TEST INFRASTRUCTURE — writes the stored per-config activation ranges of the INT8 GNN (next row NEXT-3, GNN part).

Static post-training quantisation (P:2740 calibrated the embedding the same way): the fp32 ORACLE runs on
the config's calibration events (C0 / C1: the event itself; C2, shared by C3: the first 4 events; C4: the first 2 --
the gain-calibration sample of oracle/calibrate_gain.py) and a max observer records the range of every layer's input
of every GNN MLP.  Stored as "int8_gnn_alpha" {mlp name: [one value per layer]} in
paper_2508_07423_b200/config_constants.json; nothing here touches the CUDA library.

Run:  python -m oracle.calibrate_int8_gnn
"""
from __future__ import annotations

import json
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

from oracle import etx_oracle as orc  # noqa: E402
from oracle.calibrate_gain import GAIN_EVENTS  # noqa: E402
from paper_2508_07423_b200 import synth  # noqa: E402  (input generator only)


def calibrate(name: str):
    cfg = synth.CONFIGS[name]
    batch = synth.generate_events(cfg, range(min(GAIN_EVENTS[name], cfg.n_events)))
    blob = synth.generate_weights(cfg)
    layout = {s.name: (s.dims, s.offset) for s in synth.model_layout(cfg)}
    fe, fn = orc.features(batch, synth.NORM_CENTER, synth.NORM_SCALE)
    emb = orc.mlp(fe, *layout["emb"][:1], blob, layout["emb"][1])
    src, dst = orc.build_graph(batch["event_ptr"], batch["plane"], emb, synth.r2_max(cfg), cfg.max_plane_gap)
    return orc.gnn_int8_calibration(fn, src, dst, cfg.n_iter, blob, layout)


def main():
    path = os.path.join(os.path.dirname(os.path.abspath(synth.__file__)), "config_constants.json")
    with open(path) as f:
        out = json.load(f)
    for name in ("c0", "c1", "c2", "c4"):
        out[name]["int8_gnn_alpha"] = calibrate(name)
        print(name, {k: [round(x, 3) for x in v] for k, v in out[name]["int8_gnn_alpha"].items()})
    with open(path, "w") as f:
        json.dump(out, f, indent=1, sort_keys=True)
        f.write("\n")


if __name__ == "__main__":
    main()
