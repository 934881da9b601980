"""TEST INFRASTRUCTURE — writes the stored per-config activation ranges of the INT8 embedding (next row NEXT-3).

Static post-training quantisation: a representative sample is passed through the fp32 model
and the range of every activation is recorded.  Reading (Q21): max observer; sample = the config's
calibration events (C0/C1: the event itself; C2/C4: the first 16 events; C3 shares C2's), the ORACLE's fp32
embedding MLP.  The ranges are stored next to the radius in paper_2508_07423_b200/config_constants.json
("int8_act_alpha", one value per layer input) and read by both paths; nothing here touches the CUDA library.

Run:  python -m oracle.calibrate_int8
"""
from __future__ import annotations

import json
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

from oracle import etx_oracle as orc  # noqa: E402
from paper_2508_07423_b200 import synth  # noqa: E402  (input generator only)


def calibrate(name: str):
    cfg = synth.CONFIGS[name]
    batch = synth.generate_events(cfg, range(min(cfg.calib_events, cfg.n_events)))
    blob = synth.generate_weights(cfg)
    spec = synth.model_layout(cfg)[0]
    fe, _ = orc.features(batch, synth.NORM_CENTER, synth.NORM_SCALE)
    return [float(a) for a in orc.int8_calibration(fe, spec.dims, blob, spec.offset)]


def main():
    path = os.path.join(os.path.dirname(os.path.abspath(synth.__file__)), "config_constants.json")
    with open(path) as f:
        out = json.load(f)
    for name in ("c0", "c1", "c2", "c4"):
        out[name]["int8_act_alpha"] = calibrate(name)
    with open(path, "w") as f:
        json.dump(out, f, indent=1, sort_keys=True)
        f.write("\n")
    print(json.dumps({k: v["int8_act_alpha"] for k, v in out.items()}, indent=1))


if __name__ == "__main__":
    main()
