"""The oracle against its stored trace (tests/golden/cfg0_oracle_trace.json, written by
tests/golden/make_golden.py from `oracle/` alone).  The paper prints no numbers for this path,
so the trace is a change detector: a later edit of the oracle's arithmetic shows up here and has
to be justified (passage or DESIGN.md reading) in the commit that regenerates the file.  The
GPU side of the same trace is checked in tests/test_gpu_parity.py::test_golden_trace_on_gpu."""
import importlib.util
import json
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
GOLDEN = os.path.join(HERE, "golden", "cfg0_oracle_trace.json")


def _maker():
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    return m


def test_oracle_reproduces_its_stored_trace():
    stored = json.load(open(GOLDEN))
    fresh = _maker().trace()
    assert [r["step"] for r in fresh["rows"]] == [r["step"] for r in stored["rows"]]
    for a, b in zip(fresh["rows"], stored["rows"]):
        for key in ("t1_flips", "t1_candidates", "t1_blocked", "cell_vertex_num_hist"):
            assert a[key] == b[key], (a["step"], key)
        # libm may differ in the last ulp between hosts (R16): far inside these bounds
        for key, tol in (("energy", 1e-9), ("sum_area", 1e-12), ("sum_perimeter", 1e-10), ("max_force", 1e-8),
                         ("pos_checksum", 1e-9), ("theta_sum", 1e-11)):
            assert abs(a[key] - b[key]) <= tol * max(1.0, abs(b[key])), (a["step"], key, a[key], b[key])


def test_stored_trace_obeys_the_invariants():
    """what the mathematics fixes about the stored numbers themselves"""
    stored = json.load(open(GOLDEN))
    flips = [r["t1_flips"] for r in stored["rows"]]
    assert flips == sorted(flips) and flips[-1] > 0
    for r in stored["rows"]:
        assert abs(r["sum_area"] - 64.0) <= 64.0 * 1e-12                 # total area = L^2 (L = 8)
        hist = np.array(r["cell_vertex_num_hist"])
        assert hist.sum() == 64 and (hist * np.arange(len(hist))).sum() == 6 * 64   # mean 6 sides (Euler, V = 2N)
        assert r["t1_flips"] + r["t1_blocked"] == r["t1_candidates"]
