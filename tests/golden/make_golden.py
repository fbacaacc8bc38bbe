#!/usr/bin/env python
"""Writes tests/golden/oracle_regression.json from the CPU oracle ALONE (never from the CUDA path).

The paper prints no worked numeric example for this path, so this file is not a paper value:
it freezes the oracle's output on two small seeded frames so that an unintended change of the oracle's
arithmetic shows up in `pytest -m "not gpu"`.  Run from the repo root: python tests/golden/make_golden.py
"""
import hashlib
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import oracle  # noqa: E402
from paper_1811_11481_b200 import synth  # noqa: E402  (seeded input generator only)

CASES = [dict(cfg=1, scale=0.25, seed=1), dict(cfg=2, scale=0.02, seed=2)]


def digest(case):
    fr = synth.generate(synth.config(case["cfg"], scale=case["scale"], seed=case["seed"]))
    r = oracle.track(fr.clusters, fr.sector_offsets, synth.row_x())
    h = lambda a: hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()  # noqa: E731
    return dict(case=case, n_clusters=int(fr.n), input_sha256=h(fr.clusters), n_start_hits=int(len(r.start_hits)),
                n_tracks=int(len(r.tracks)), link_up_sha256=h(r.link_up), start_hits_sha256=h(r.start_hits),
                assignment_sha256=h(r.assignment), tracks_sha256=h(r.tracks),
                first_track=[float(r.tracks[f][0]) for f in ("x", "y", "z", "sinphi", "dzds", "qpt", "chi2")])


if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_regression.json")
    json.dump([digest(c) for c in CASES], open(out, "w"), indent=1)
    print("wrote", out)
