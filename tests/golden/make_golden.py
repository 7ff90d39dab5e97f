"""Writes tests/golden/*.json from the CPU oracle ONLY (never from the CUDA path).

Run:  python tests/golden/make_golden.py
The paper prints no worked example with numbers (PAPER.md gives the method in words and
its figures are missing), so these files are regression pins of the oracle itself on the
seeded BASELINE.json configs[0] event and on one hand-made track: they make a later
change to the oracle's arithmetic visible.  The independent pins are in
tests/test_oracle_pins.py.
"""
import hashlib
import json
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "oracle"))
import hough_oracle as oracle  # noqa: E402
from paper_1305_4855_b200 import synth  # noqa: E402


def record(grid, x, y, layer):
    r = oracle.run(grid, x, y, layer)
    return {
        "hits_sha256": synth.event_sha256(x, y, layer),
        "n_hits": int(len(x)),
        "n_votes": r["n_votes"],
        "acc_sha256": hashlib.sha256(r["acc"].tobytes()).hexdigest(),
        "peak_bin": r["peak_bin"].tolist(),
        "peak_mask": r["peak_mask"].tolist(),
        "hit_offset": r["hit_offset"].tolist(),
        "hit_index": r["hit_index"].tolist(),
    }


def main():
    w = synth.WORKLOADS["prompt2d"]
    x, y, layer, _ = synth.generate_event(w.event, 0)
    out = {"cite": "BASELINE.json configs[0], seed 0; oracle = SURVEY.md 8(c) A1-A7",
           "prompt2d_seed0": record(w.grid, x, y, layer)}
    g = synth.Grid(n_phi=64, n_d0=16, n_kappa=64, L_min=9)
    x, y, layer = synth.single_track_event(g, 21, 9, 0.0033)
    out["single_track_64x16x64_i21_j9_k0.0033"] = record(g, x, y, layer)
    with open(os.path.join(HERE, "oracle_regression.json"), "w") as f:
        json.dump(out, f, indent=1)


if __name__ == "__main__":
    main()
