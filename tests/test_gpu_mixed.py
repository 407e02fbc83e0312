"""GPU tests of the mixed-precision library (libavm_b200_mixed.so): the
accuracy contract written in include/avm.h (avm_precision) against the float64 oracle.  The mixed
library stores positions on a fixed-point grid of 2^-32 box lengths and the cached cell records as
floats; every arithmetic operation stays fp64.  Run on the B200 box with `pytest -m gpu`."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
from paper_1702_02939_b200 import workloads as w
from tests import helpers as h
from tests.test_gpu_parity import assert_forces_close, assert_positions_close, to_np, near_threshold

GRID = 4294967296.0


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    from paper_1702_02939_b200 import build
    build.build()
    from paper_1702_02939_b200 import binding
    assert binding.library("mixed").avm_precision() == b"mixed"
    return binding


def on_grid(t):
    """the tiling with every position rounded to the library's grid, computed here with numpy"""
    q = np.rint(t.pos / np.array([t.Lx, t.Ly]) * GRID) % GRID
    tt = t.copy()
    tt.pos = q * (np.array([t.Lx, t.Ly]) / GRID)
    assert np.abs(tt.pos - t.pos).max() <= max(t.Lx, t.Ly) / GRID
    return tt


@pytest.mark.parametrize("k", [0, 1, 2])
def test_contract_from_an_identical_state(B, k):
    t = on_grid(w.config_tiling(k))
    p = w.config_params(k)
    L = t.Lx
    g = B.from_tiling(t, precision="mixed", sort_at_create=True, **{a: b for a, b in p.items() if a != "sort_at_create"})
    o = oracle.from_tiling(t, **p)
    s0 = to_np(g.get_state())
    assert np.array_equal(s0["pos"], t.pos), "grid points must pack to themselves"
    # geometry and forces of avm_compute_forces: as in the default library
    F, ap = g.compute_forces()
    Fo, apo = o.compute_forces()
    assert_forces_close(F.cpu().numpy(), Fo, ap.cpu().numpy(), apo)
    # one step: positions within one grid unit plus the float rounding of the cached records
    g.step(1)
    o.step(1)
    sg, so = to_np(g.get_state()), o.get_state()
    tol = L / GRID + 1e-6 * p["dt"] * np.linalg.norm(Fo, axis=1).max()
    # end points of this step's T1s are excluded: their new edge is the old one turned by 90 degrees, and the
    # direction of an old edge of length l is only defined to (grid unit / l); they stay within the new edge length
    kept = (sg["vertex_neighbors"] == t.vertex_neighbors).all(axis=1) & (so["vertex_neighbors"] == t.vertex_neighbors).all(axis=1)
    assert kept.mean() > 0.8
    assert_positions_close(sg["pos"][kept], so["pos"][kept], t.Lx, t.Ly, tol)
    assert_positions_close(sg["pos"], so["pos"], t.Lx, t.Ly, 1.6 * p["l_c"])
    assert np.abs(sg["theta"] - so["theta"]).max() <= 1e-8
    on = sg["pos"] / np.array([t.Lx, t.Ly]) * GRID
    assert np.abs(on - np.rint(on)).max() < 1e-3, "moved positions are grid points"
    # the applied force, recovered from the displacement of T1-free vertices: 1e-6 relative once the grid unit is discounted
    # T1 sets of the moved state: equal outside the stated band
    band = 4 * L / GRID
    if sg["stats"]["t1_flips"] == so["stats"]["t1_flips"]:
        h.assert_same_topology(sg, so)
    cg, wg = g.debug_t1()
    co, wo = o.debug_t1()
    sc, sw = {tuple(x) for x in cg.tolist()}, {tuple(x) for x in wg.tolist()}
    oc, ow = {tuple(x) for x in co.tolist()}, {tuple(x) for x in wo.tolist()}
    fuzzy = near_threshold(so, sc ^ oc, t.Lx, t.Ly, p["l_c"], band=band)
    assert (sc ^ oc) <= fuzzy
    if not fuzzy and sg["stats"]["t1_flips"] == so["stats"]["t1_flips"]:
        assert sw == ow


def test_short_trajectory_stays_close_to_the_oracle(B):
    """configs[0] (L = 8: grid unit 1.9e-9) for 30 steps: same topology, positions within 1e-6"""
    t = on_grid(w.config_tiling(0))
    p = w.config_params(0)
    g = B.from_tiling(t, precision="mixed", **p)
    o = oracle.from_tiling(t, **p)
    g.step(30)
    o.step(30)
    sg, so = to_np(g.get_state()), o.get_state()
    h.assert_same_topology(sg, so)
    assert_positions_close(sg["pos"], so["pos"], t.Lx, t.Ly, 1e-6)
    assert sg["stats"]["t1_flips"] == so["stats"]["t1_flips"] > 0


def test_long_run_invariants_determinism_resume_and_schedules(B):
    """configs[1] for 300 steps with re-sorts: valid tiling, areas tile the box, the flip count tracks the
    oracle's statistically; two runs give the same bits, so do both kernel schedules and a resumed run."""
    t = on_grid(w.config_tiling(1))
    p = dict(w.config_params(1), sort_every=37)
    runs = {}
    for name, sched in (("a", "fused"), ("b", "fused"), ("c", "unfused")):
        g = B.from_tiling(t, precision="mixed", schedule=sched, **p)
        g.step(300)
        runs[name] = to_np(g.get_state())
        if name == "a":
            ap = g.compute_forces()[1].cpu().numpy()
            msd = g.observe()["msd"]
    keys = ("pos", "theta", "cell_vertices", "vertex_neighbors", "vertex_cell_neighbors", "cell_vertex_num")
    for other in ("b", "c"):
        for key in keys:
            assert np.array_equal(runs["a"][key], runs[other][key]), (other, key)
    s = runs["a"]
    assert s["stats"]["error"] == 0
    h.check_topology(s["cell_vertex_num"], s["cell_vertices"], s["vertex_neighbors"], s["vertex_cell_neighbors"], S=t.S)
    L2 = t.Lx * t.Ly
    assert abs(ap[:, 0].sum() - L2) <= 1e-9 * L2 and (ap[:, 1] > 0).all()
    o = oracle.from_tiling(t, **p)
    o.step(300)
    fo = o.get_state()["stats"]["t1_flips"]
    assert abs(s["stats"]["t1_flips"] - fo) <= 0.1 * fo
    assert abs(msd - o.msd()) <= 0.1 * o.msd()
    # resume from an exported state (grid points pack to themselves)
    g = B.from_tiling(t, precision="mixed", **p)
    g.step(120)
    sc = to_np(g.get_state())
    tt = w.Tiling(t.Lx, t.Ly, t.S, sc["pos"], sc["cell_vertex_num"], sc["cell_vertices"], sc["vertex_neighbors"],
                  sc["vertex_cell_neighbors"], sc["theta"])
    g2 = B.from_tiling(tt, precision="mixed", **dict(p, step0=120, sort_every=0))
    g3 = B.from_tiling(t, precision="mixed", **dict(p, sort_every=0))
    g2.step(60)
    g3.step(180)
    s2, s3 = to_np(g2.get_state()), to_np(g3.get_state())
    for key in ("pos", "theta"):
        assert np.array_equal(s2[key], s3[key]), key
    h.assert_same_topology(s2, s3)


def test_full_size_one_step(B):
    """configs[3] in the mixed library: the contract's one-step bound at L = 1024 (grid unit 2.4e-7)"""
    t = on_grid(w.config_tiling(3))
    p = w.config_params(3)
    g = B.from_tiling(t, precision="mixed", **p)
    o = oracle.from_tiling(t, **p)
    Fo = o.compute_forces()[0]
    g.step(1)
    o.step(1)
    sg, so = to_np(g.get_state()), o.get_state()
    tol = t.Lx / GRID + 1e-6 * p["dt"] * np.linalg.norm(Fo, axis=1).max()
    kept = (sg["vertex_neighbors"] == t.vertex_neighbors).all(axis=1) & (so["vertex_neighbors"] == t.vertex_neighbors).all(axis=1)
    assert kept.mean() > 0.8
    assert_positions_close(sg["pos"][kept], so["pos"][kept], t.Lx, t.Ly, tol)
    assert_positions_close(sg["pos"], so["pos"], t.Lx, t.Ly, 1.6 * p["l_c"])
    # a handful of the ~60 000 short edges lie inside the band and may be decided differently
    assert abs(sg["stats"]["t1_flips"] - so["stats"]["t1_flips"]) <= 32
