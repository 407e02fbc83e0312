"""Writes tests/golden/cfg0_oracle_trace.json: a trace of the CPU oracle on configs[0]
(BASELINE.json: N = 64 cells, L = 8, Voronoi seed 1, Philox seed 7, 100 steps).

    python tests/golden/make_golden.py

The values come from `oracle/` only (plus the seeded input generator both sides share); nothing
here touches the CUDA path.  The paper (arXiv:1702.02939) prints no trajectory, energy trace or
T1 count, so this file is a change detector for the oracle's arithmetic, not a pin to the paper:
the pins proper are the invariants in tests/test_oracle_*.py.  A commit that changes this file
must name the passage or DESIGN.md reading that justifies the change.
"""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import numpy as np

import oracle
from paper_1702_02939_b200 import workloads as w


def trace():
    t = w.config_tiling(0)
    p = w.config_params(0)
    o = oracle.from_tiling(t, **p)
    rows = []
    for step in (0, 1, 2, 5, 10, 20, 50, 100):
        o.step(step - o.get_state()["stats"]["step"])
        s = o.get_state()
        F, ap = o.compute_forces()
        rows.append({
            "step": step,
            "energy": float(o.energy()),
            "sum_area": float(ap[:, 0].sum()),
            "sum_perimeter": float(ap[:, 1].sum()),
            "max_force": float(np.linalg.norm(F, axis=1).max()),
            "pos_checksum": float((s["pos"] * np.arange(1, 2 * t.V + 1).reshape(t.V, 2)).sum()),
            "theta_sum": float(s["theta"].sum()),
            "t1_flips": int(s["stats"]["t1_flips"]),
            "t1_candidates": int(s["stats"]["t1_candidates"]),
            "t1_blocked": int(s["stats"]["t1_blocked"]),
            "cell_vertex_num_hist": np.bincount(s["cell_vertex_num"], minlength=17).tolist(),
        })
    return {"config": "BASELINE.json configs[0]", "source": "oracle/avm_oracle.cpp via tests/golden/make_golden.py",
            "rows": rows}


if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg0_oracle_trace.json")
    with open(out, "w") as f:
        json.dump(trace(), f, indent=1)
    print("wrote", out)
