"""TEST INFRASTRUCTURE — writes the stored per-config weight gain g (SURVEY.md Q14 / DESIGN.md readings).

The thesis trains its networks; BASELINE.json only says "Xavier init from seed".  With untrained
Xavier weights the residual message passing either collapses every score onto one value or saturates them,
so the input recipe carries ONE gain g on the last layer of every node / edge network phi_k, psi_k.
SURVEY Q14 fixes how g is chosen, and it is an ORACLE-side criterion (nothing here touches the CUDA library,
and no GPU error enters the choice):

    start at g = 0.25 and take the SMALLEST g on the grid 0.25, 0.30, 0.35, ... , 1.50 at which, on the
    config's gain-calibration events scored by the fp64-accumulating oracle,
      (i)   at least 50 % of the edge scores fall in (0.02, 0.98)            (not saturated),
      (ii)  max |h| < 1e3 and max |e| < 1e3 over every message-passing step's final state,
      (iii) the standard deviation of the scores is at least STD_FLOOR = 0.05 (not collapsed: the 1e-4 / 2e-2
            score gates must look at scores that actually differ from edge to edge).

Gain-calibration events: C0 / C1 the event itself; C2 (and C3, which shares C2's stream) the first 4 events;
C4 the first 2 events (the oracle needs seconds per event).  The graph is the oracle's own graph at the
stored radius, so oracle/calibrate_radius.py must have run first.

The result is stored as "gain" (with the statistics that justified it, and the statistics of every grid value
tried) in paper_2508_07423_b200/config_constants.json; synth.generate_weights reads it from there.

Run:  python -m oracle.calibrate_gain            (writes the constants)
      python -m oracle.calibrate_gain --table    (prints the statistics over the whole grid, writes nothing)
"""
from __future__ import annotations

import dataclasses
import json
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

from oracle import etx_oracle as orc  # noqa: E402
from paper_2508_07423_b200 import synth  # noqa: E402  (input generator only)

GRID = [round(0.25 + 0.05 * i, 2) for i in range(26)]     # 0.25 .. 1.50
STD_FLOOR = 0.05
FRAC_MIN = 0.5
ABS_MAX = 1e3
GAIN_EVENTS = {"c0": 1, "c1": 1, "c2": 4, "c4": 2}


def stats(name: str, g: float) -> dict:
    """Oracle statistics of the config's gain-calibration events with gain g."""
    cfg = dataclasses.replace(synth.CONFIGS[name], gain=g)
    batch = synth.generate_events(cfg, range(min(GAIN_EVENTS[name], cfg.n_events)))
    blob = synth.generate_weights(cfg)
    layout = {s.name: (s.dims, s.offset) for s in synth.model_layout(cfg)}
    out = orc.run_path(batch, blob, layout, cfg.gnn_hidden, cfg.n_iter, synth.r2_max(cfg), cfg.max_plane_gap,
                       synth.NORM_CENTER, synth.NORM_SCALE)
    s = out["scores"].astype(np.float64)
    return {"gain": g, "n_edges": int(len(s)), "score_std": float(s.std()),
            "frac_unsaturated": float(np.mean((s > 0.02) & (s < 0.98))),
            "score_min": float(s.min()), "score_max": float(s.max()),
            "max_abs_h": float(np.abs(out["h"]).max()), "max_abs_e": float(np.abs(out["e"]).max())}


def accept(st: dict) -> bool:
    return (st["frac_unsaturated"] >= FRAC_MIN and st["max_abs_h"] < ABS_MAX and st["max_abs_e"] < ABS_MAX
            and st["score_std"] >= STD_FLOOR)


def calibrate(name: str) -> dict:
    tried = []
    for g in GRID:
        st = stats(name, g)
        tried.append(st)
        if accept(st):
            return {"gain": g, "gain_stats": st, "gain_tried": tried,
                    "gain_rule": f"smallest g in 0.25(0.05)1.50 with frac(0.02<s<0.98)>={FRAC_MIN}, "
                                 f"max|h|,|e|<{ABS_MAX:g}, std(s)>={STD_FLOOR}"}
    raise RuntimeError(f"{name}: no gain on the grid satisfies SURVEY Q14's criterion")


def main():
    path = os.path.join(os.path.dirname(os.path.abspath(synth.__file__)), "config_constants.json")
    if "--table" in sys.argv:
        for name in ("c0", "c1", "c2", "c4"):
            for g in GRID[:16]:
                st = stats(name, g)
                print(name, json.dumps(st), "ACCEPT" if accept(st) else "")
        return
    with open(path) as f:
        out = json.load(f)
    for name in ("c0", "c1", "c2", "c4"):
        out[name].update(calibrate(name))
        print(name, out[name]["gain"], json.dumps(out[name]["gain_stats"]))
    with open(path, "w") as f:
        json.dump(out, f, indent=1, sort_keys=True)
        f.write("\n")


if __name__ == "__main__":
    main()
