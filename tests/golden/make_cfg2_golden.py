"""Writes tests/golden/cfg2_full_oracle.json: the CPU oracle's result for BASELINE config 2 (6-D
Lorenz '96 headline run to t = 0.5, prune every 5 steps) at full size. Calls ONLY oracle/ (plus the
seeded workload parameters). Takes several minutes on one core.

    python tests/golden/make_cfg2_golden.py
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle.binding import Oracle  # noqa: E402
from paper_2508_13986_b200 import workloads as W  # noqa: E402


def main():
    cfg = W.config2()
    o = Oracle(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"])
    o.init_gaussian(cfg["mean"], cfg["cov"])
    k, counts, dts = 0, [o.count()], []
    while o.time() < cfg["t_end"]:
        dts.append(o.step(cfg["t_end"] - o.time()))
        k += 1
        if k % cfg["prune_every"] == 0:
            o.prune()
        counts.append(o.count())
    keys, p = o.export()          # sorted lexicographically
    rng = np.random.default_rng(W.S0 + 22)
    top = np.argsort(-p)[:32]     # the 32 heaviest cells
    rnd = rng.choice(len(p), 96, replace=False)
    idx = np.unique(np.concatenate([top, rnd]))
    out = {
        "citation": "BASELINE.json configs[2]; oracle = oracle/gbees_oracle.cpp (DESIGN.md D1-D5)",
        "steps": k, "t": o.time(), "final_cells": int(len(p)), "cells_after_each_step": [int(c) for c in counts],
        "dt_first": dts[0], "dt_last": dts[-1], "p_max": float(p.max()),
        "sample_keys": keys[idx].tolist(), "sample_p": [float(v) for v in p[idx]],
    }
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg2_full_oracle.json")
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
    print("wrote", path, "steps", k, "cells", len(p))


if __name__ == "__main__":
    main()
