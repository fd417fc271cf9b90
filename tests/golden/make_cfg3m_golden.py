"""Writes tests/golden/cfg3m_full_oracle.json: the CPU oracle's result for a mid-scale twin of
BASELINE config 3 (linear 6-D stress f = Ax, dx = 0.7, all 50 steps, prune every 5; about 1 M cells:
the largest size the serial oracle finishes in tens of minutes -- the 1/10-scale twin (dx = 0.5,
10 M cells) needs ~5 minutes per oracle step). Calls ONLY oracle/ (plus the seeded workload parameters).

    python tests/golden/make_cfg3m_golden.py
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
    cfg = W.config3(dx=0.7)
    o = Oracle(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"])
    o.init_gaussian(cfg["mean"], cfg["cov"])
    k, counts, dts = 0, [o.count()], []
    while k < cfg["steps"]:
        dts.append(o.step())
        k += 1
        print("step", k, "cells", o.count(), flush=True)
        if k % cfg["prune_every"] == 0:
            o.prune()
        counts.append(o.count())
    keys, p = o.export()          # sorted lexicographically
    rng = np.random.default_rng(W.S0 + 22)
    top = np.argsort(-p)[:32]     # the 32 heaviest cells
    rnd = rng.choice(len(p), 96, replace=False)
    idx = np.unique(np.concatenate([top, rnd]))
    out = {
        "citation": "BASELINE.json configs[3] with dx = 0.7 (mid-scale twin); oracle = oracle/gbees_oracle.cpp (DESIGN.md D1-D5)",
        "steps": k, "t": o.time(), "final_cells": int(len(p)), "cells_after_each_step": [int(c) for c in counts],
        "dt_first": dts[0], "dt_last": dts[-1], "p_max": float(p.max()),
        "sample_keys": keys[idx].tolist(), "sample_p": [float(v) for v in p[idx]],
    }
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg3m_full_oracle.json")
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
    print("wrote", path, "steps", k, "cells", len(p))


if __name__ == "__main__":
    main()
