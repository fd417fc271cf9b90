"""Writes tests/golden/cfg3s_full_oracle.json: the CPU oracle's result for the 1/10-scale twin of
BASELINE config 3 (linear 6-D stress f = Ax, dx = 0.5, all 50 steps, prune every 5; 6 M -> 10 M cells;
SURVEY.md 8(d) "full 50 steps on a 1/10-scale twin"). Calls ONLY oracle/ (plus the seeded workload
parameters). Takes several HOURS on one core (about 5 minutes per step); the file is rewritten after
every prune so that a partial run is still usable (the GPU test compares as many prunes as are stored).

Stored, after every prune and at the end: the cell count and sha256 of the int32 key array sorted
lexicographically (bit-exact active-set check); at the end also 4096 sampled masses, the six 1-D
marginals and the first two moments in index units.

    python tests/golden/make_cfg3s_golden.py
"""
import hashlib
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle.binding import Oracle  # noqa: E402
from paper_2508_13986_b200 import workloads as W  # noqa: E402


def sorted_state(keys, p):
    """Lexicographic order (dim 0 most significant) through one packed int64 sort key (|c| < 2^9)."""
    code = np.zeros(len(keys), dtype=np.int64)
    for j in range(keys.shape[1]):
        code = (code << 10) | (keys[:, j].astype(np.int64) + 512)
    order = np.argsort(code, kind="stable")
    return np.ascontiguousarray(keys[order]), p[order]


def key_hash(keys_sorted):
    return hashlib.sha256(np.ascontiguousarray(keys_sorted, dtype=np.int32).tobytes()).hexdigest()


def main():
    cfg = W.config3(dx=0.5)
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg3s_full_oracle.json")
    o = Oracle(cfg["n"], cfg["dx"], cfg["thresh"], cfg["dyn"], cfg["params"], cfl=cfg["cfl"])
    o.init_gaussian(cfg["mean"], cfg["cov"])
    out = {"citation": "BASELINE.json configs[3] at 1/10 scale (dx = 0.5; SURVEY.md 8(d)); oracle = oracle/gbees_oracle.cpp (DESIGN.md D1-D5)",
           "cells_initial": o.count(), "after_prune": {}, "dts": []}
    t0 = time.time()
    k = 0
    while k < cfg["steps"]:
        out["dts"].append(o.step())
        k += 1
        print("step", k, "cells", o.count(), f"{time.time() - t0:.0f} s", flush=True)
        if k % cfg["prune_every"] == 0:
            o.prune()
            keys, p = o.export(sort=False)
            ks, ps = sorted_state(keys, p)
            out["after_prune"][str(k)] = {"cells": int(len(ps)), "keys_sha256": key_hash(ks), "t": o.time(),
                                          "p_max": float(ps.max())}
            if k == cfg["steps"]:
                rng = np.random.default_rng(W.S0 + 33)
                idx = np.unique(np.concatenate([np.argsort(-ps)[:64], rng.choice(len(ps), 4032, replace=False)]))
                x = ks.astype(np.float64)
                mean = ps @ x
                d = x - mean
                out["final"] = {
                    "steps": k, "t": o.time(), "cells": int(len(ps)), "keys_sha256": key_hash(ks), "p_max": float(ps.max()),
                    "sample_keys": ks[idx].tolist(), "sample_p": [float(v) for v in ps[idx]],
                    "mean_index_units": mean.tolist(), "cov_index_units": (d.T @ (d * ps[:, None])).tolist(),
                    "marginals_1d": [{"coords": np.unique(ks[:, j]).tolist(),
                                      "mass": np.bincount(np.unique(ks[:, j], return_inverse=True)[1], weights=ps).tolist()}
                                     for j in range(ks.shape[1])]}
            with open(path, "w") as f:
                json.dump(out, f, indent=1)
            print("wrote", path, "through step", k, flush=True)


if __name__ == "__main__":
    main()
