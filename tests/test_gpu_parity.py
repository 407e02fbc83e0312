"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by element
on the same seeded inputs.  Tolerances are BASELINE.json's `north_star`:
  * per-step geometry and forces from an identical state: 1e-10 relative (fp64);
  * T1 candidate sets and post-flip topology: bit-exact in canonical form (R19), excluding edges
    within 1e-9 of l_c;
  * trajectories: 1e-8 in positions over the first 100 steps of configs[0].
Run on the B200 box with `pytest -m gpu`."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
from paper_1702_02939_b200 import workloads as w
from tests import helpers as h


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    from paper_1702_02939_b200 import build
    build.build()
    from paper_1702_02939_b200 import binding
    return binding


_TILINGS = {}


def tiling(k):
    if k not in _TILINGS:
        _TILINGS[k] = w.config_tiling(k)
    return _TILINGS[k]


def to_np(state):
    return {k: (v.cpu().numpy() if hasattr(v, "cpu") else v) for k, v in state.items()}


def assert_forces_close(F, Fo, ap, apo):
    # per-cell relative on A and P (areas can be tiny/negative transiently: guard with mean scale)
    sa = np.maximum(np.abs(apo[:, 0]), np.abs(apo[:, 0]).mean())
    assert (np.abs(ap[:, 0] - apo[:, 0]) <= 1e-10 * sa).all()
    assert (np.abs(ap[:, 1] - apo[:, 1]) <= 1e-10 * np.abs(apo[:, 1])).all()
    rms = np.sqrt((Fo ** 2).sum(axis=1).mean())
    nf = np.linalg.norm(Fo, axis=1)
    err = np.linalg.norm(F - Fo, axis=1)
    assert (err <= 1e-10 * np.maximum(nf, rms)).all(), (err / np.maximum(nf, rms)).max()


def assert_positions_close(p, po, Lx, Ly, tol):
    d = p - po
    d = np.hypot(h.min_image(d[:, 0], Lx), h.min_image(d[:, 1], Ly))
    assert d.max() <= tol, d.max()


def assert_states_match(sg, so, Lx, Ly, pos_tol=1e-8):
    h.assert_same_topology(sg, so)
    assert_positions_close(sg["pos"], so["pos"], Lx, Ly, pos_tol)
    assert np.abs(sg["theta"] - so["theta"]).max() <= pos_tol
    for key in ("step", "t1_short", "t1_candidates", "t1_flips", "t1_blocked", "overflow_rejects", "error"):
        assert sg["stats"][key] == so["stats"][key], key


# ------------------------------------------------------------------------------------------------
def test_philox_words_bit_exact(B):
    t = tiling(0)
    sim = B.from_tiling(t, **w.config_params(0))
    for seed, step, cell0 in [(7, 0, 0), (7, 99, 1000), (0xDEADBEEFCAFEF00D, (3 << 32) | 17, 2 ** 31 - 5000)]:
        got = sim.philox_words(seed, step, cell0, 4096)
        assert np.array_equal(got, oracle.philox_words(seed, step, cell0, 4096))


@pytest.mark.parametrize("k", [0, 1, 2])
@pytest.mark.parametrize("sort", [False, True])
def test_geometry_and_forces_parity(B, k, sort):
    t = tiling(k)
    p = dict(w.config_params(k), sort_at_create=sort)
    sim = B.from_tiling(t, **p)
    F, ap = sim.compute_forces()
    Fo, apo = oracle.from_tiling(t, **p).compute_forces()
    assert_forces_close(F.cpu().numpy(), Fo, ap.cpu().numpy(), apo)
    assert abs(sim.energy() - oracle.from_tiling(t, **p).energy()) <= 1e-11 * abs(oracle.from_tiling(t, **p).energy())
    # host-pointer twin gives the same bits
    Fh, aph = sim.compute_forces_host()
    assert np.array_equal(Fh, F.cpu().numpy()) and np.array_equal(aph, ap.cpu().numpy())


def test_hexagons_have_zero_force_on_gpu(B):
    t = w.hex_tiling(8, 6, a=0.62)
    sim = B.from_tiling(t, KA=1.3, KP=0.7, A0=1.0, P0=3.6)
    F, ap = sim.compute_forces()
    assert F.abs().max().item() <= 1e-12
    assert np.allclose(ap.cpu().numpy()[:, 0], 1.5 * np.sqrt(3) * 0.62 ** 2, rtol=1e-13)


def test_trajectory_parity_cfg0_100_steps(B):
    """The headline trajectory bar: 100 steps of configs[0], positions within 1e-8 at EVERY step,
    topology and T1 counters bit-exact, through the step-0 T1 burst."""
    t = tiling(0)
    p = w.config_params(0)
    g = B.from_tiling(t, **p)
    o = oracle.from_tiling(t, **p)
    for s in range(100):
        g.step(1)
        o.step(1)
        assert_states_match(to_np(g.get_state()), o.get_state(), t.Lx, t.Ly)
    st = g.stats()
    assert st["t1_flips"] > 0 and st["error"] == 0


@pytest.mark.parametrize("k,steps,chunk", [(1, 60, 10), (2, 12, 4)])
def test_trajectory_parity_larger_configs(B, k, steps, chunk):
    t = tiling(k)
    p = w.config_params(k)
    g = B.from_tiling(t, **p)
    o = oracle.from_tiling(t, **p)
    for s in range(0, steps, chunk):
        g.step(chunk)
        o.step(chunk)
        assert_states_match(to_np(g.get_state()), o.get_state(), t.Lx, t.Ly)
    assert g.stats()["t1_flips"] > 50


@pytest.mark.parametrize("sched", ["fused", "unfused", "persistent"])
@pytest.mark.parametrize("k,steps,chunk", [(0, 100, 5), (1, 40, 10)])
def test_trajectory_parity_with_mobility_and_moduli_other_than_one(B, k, steps, chunk, sched):
    """every other dynamic test runs mu = K_A = K_P = A0 = 1, where a dropped or misplaced factor in the
    move (Eq. 4) or in the force prefactors (Eq. A1-A3) would go unnoticed.  Same bar as
    the headline trajectory test, through the T1 burst, in every schedule."""
    t = tiling(k)
    p = dict(w.config_params(k), mu=0.6, KA=1.7, KP=0.6, A0=1.2)
    g = B.from_tiling(t, schedule=sched, **p)
    o = oracle.from_tiling(t, **p)
    for s in range(0, steps, chunk):
        g.step(chunk)
        o.step(chunk)
        assert_states_match(to_np(g.get_state()), o.get_state(), t.Lx, t.Ly)
    st = g.stats()
    assert st["t1_flips"] >= 20 and st["error"] == 0


@pytest.mark.parametrize("sched", ["fused", "unfused", "persistent"])
def test_an_edge_whose_end_cells_coincide_does_not_flip_on_gpu(B, sched):
    """GPU twin of tests/test_oracle_t1.py::test_an_edge_whose_end_cells_coincide_does_not_flip (R10, "the four cells
    are distinct"): the tiling of tests/horseshoe.py passes avm_create's validation, its one short edge is counted and
    is no candidate, neither in the test hooks nor in the cell pass of a real step (nothing moves: dt = 0)."""
    from tests import horseshoe as hs
    t, edge = hs.build()
    g = B.from_tiling(t, schedule=sched, **hs.PARAMS)
    o = oracle.from_tiling(t, **hs.PARAMS)
    cand, win = g.debug_t1()
    assert len(cand) == 0 and len(win) == 0
    g.t1_pass()
    o.t1_pass()
    assert_states_match(to_np(g.get_state()), o.get_state(), t.Lx, t.Ly, pos_tol=0.0)
    g.step(3)
    o.step(3)
    sg = to_np(g.get_state())
    assert_states_match(sg, o.get_state(), t.Lx, t.Ly, pos_tol=0.0)
    assert sg["stats"]["t1_short"] == 4 and sg["stats"]["t1_candidates"] == 0 and sg["stats"]["t1_flips"] == 0
    assert np.array_equal(sg["cell_vertices"], t.cell_vertices)


def near_threshold(state, pairs, Lx, Ly, l_c, band=1e-9):
    pos = state["pos"]
    out = set()
    for a, b in pairs:
        d = pos[b] - pos[a]
        l = np.hypot(h.min_image(d[0], Lx), h.min_image(d[1], Ly))
        if abs(l - l_c) < band:
            out.add((a, b))
    return out


@pytest.mark.parametrize("k,harvest", [(0, [0, 1, 3, 10]), (1, [0, 1, 2, 5, 20]), (2, [0, 2])])
def test_t1_sets_and_post_flip_topology_from_identical_states(B, k, harvest):
    """States harvested from the oracle trajectory (including the step-0 burst) are loaded into the
    CUDA path; candidate and winner sets must be equal as sets of (tag_min, tag_max), and one T1
    pass from that state must give the identical topology."""
    t = tiling(k)
    p = w.config_params(k)
    o = oracle.from_tiling(t, **p)
    done = 0
    for target in harvest:
        o.step(target - done)
        done = target
        so = o.get_state()
        tt = w.Tiling(t.Lx, t.Ly, t.S, so["pos"], so["cell_vertex_num"], so["cell_vertices"],
                      so["vertex_neighbors"], so["vertex_cell_neighbors"], so["theta"])
        for sort in (False, True):
            g = B.from_tiling(tt, **dict(p, step0=target, sort_at_create=sort))
            cand, win = g.debug_t1()
            co, wo = o.debug_t1()
            cg, wg = {tuple(x) for x in cand.tolist()}, {tuple(x) for x in win.tolist()}
            cs, ws = {tuple(x) for x in co.tolist()}, {tuple(x) for x in wo.tolist()}
            fuzzy = near_threshold(so, cg ^ cs, t.Lx, t.Ly, p["l_c"])
            assert (cg ^ cs) <= fuzzy, f"candidate sets differ at step {target}"
            if not fuzzy:
                assert wg == ws, f"winner sets differ at step {target}"
            # one pass from the identical state
            o2 = oracle.OracleSim(so["pos"], so["cell_vertex_num"], so["cell_vertices"], so["vertex_neighbors"],
                                  so["vertex_cell_neighbors"], so["theta"], **dict(p, step0=target))
            o2.t1_pass()
            g.t1_pass()
            sg, s2 = to_np(g.get_state()), o2.get_state()
            if not fuzzy:
                h.assert_same_topology(sg, s2)
                assert_positions_close(sg["pos"], s2["pos"], t.Lx, t.Ly, 1e-12)
                for key in ("t1_short", "t1_candidates", "t1_flips", "t1_blocked", "overflow_rejects"):
                    assert sg["stats"][key] == s2["stats"][key], key
            h.check_topology(sg["cell_vertex_num"], sg["cell_vertices"], sg["vertex_neighbors"],
                             sg["vertex_cell_neighbors"]) if k < 2 else None


def test_hilbert_resort_is_a_noop_in_canonical_form(B):
    t = tiling(1)
    p = w.config_params(1)
    g = B.from_tiling(t, **p)
    g.step(7)
    before = to_np(g.get_state())
    F0, ap0 = g.compute_forces()
    g.resort()
    after = to_np(g.get_state())
    h.assert_same_topology(before, after)
    assert np.array_equal(before["pos"], after["pos"]) and np.array_equal(before["theta"], after["theta"])
    F1, ap1 = g.compute_forces()
    assert (F0 - F1).abs().max().item() <= 1e-13 and (ap0 - ap1).abs().max().item() <= 1e-13
    assert after["stats"]["n_sorts"] == 1
    # sorting twice changes nothing either
    g.resort()
    again = to_np(g.get_state())
    h.assert_same_topology(before, again)


def test_sort_every_trajectory_equals_unsorted(B):
    t = tiling(1)
    p = w.config_params(1)
    a = B.from_tiling(t, **dict(p, sort_every=0))
    b = B.from_tiling(t, **dict(p, sort_every=5, sort_at_create=True))
    a.step(40)
    b.step(40)
    sa, sb = to_np(a.get_state()), to_np(b.get_state())
    h.assert_same_topology(sa, sb)
    assert_positions_close(sa["pos"], sb["pos"], t.Lx, t.Ly, 1e-8)
    assert sb["stats"]["n_sorts"] == 9 and sa["stats"]["t1_flips"] == sb["stats"]["t1_flips"]


def test_hilbert_sort_improves_locality(B):
    """After the sort, vertices of a cell and neighbours of a vertex are close in memory; checked
    through the Hilbert keys of the device function on the sorted positions."""
    t = tiling(2)
    g = B.from_tiling(t, **w.config_params(2))
    m = 9
    gx = np.minimum((t.pos[:, 0] / t.Lx * (1 << m)).astype(np.int64), (1 << m) - 1)
    gy = np.minimum((t.pos[:, 1] / t.Ly * (1 << m)).astype(np.int64), (1 << m) - 1)
    keys = g.hilbert_index(m, gx, gy)
    host = np.array([B.hilbert_index_host(m, int(x), int(y)) for x, y in zip(gx[:2000], gy[:2000])], dtype=np.uint32)
    assert np.array_equal(keys[:2000], host)
    order = np.argsort(keys, kind="stable")
    rank = np.empty_like(order)
    rank[order] = np.arange(order.size)
    nb = t.vertex_neighbors
    spread_sorted = np.abs(rank[nb] - rank[:, None]).mean()
    spread_unsorted = np.abs(nb - np.arange(t.V)[:, None]).mean()
    assert spread_sorted < 0.05 * spread_unsorted


def test_resume_and_determinism(B):
    t = tiling(1)
    p = w.config_params(1)
    a = B.from_tiling(t, **p)
    a.step(30)
    sa = to_np(a.get_state())
    b = B.from_tiling(t, **p)
    b.step(30)
    sb = to_np(b.get_state())
    for key in ("pos", "theta", "cell_vertices", "vertex_neighbors", "vertex_cell_neighbors", "cell_vertex_num"):
        assert np.array_equal(sa[key], sb[key]), f"run-to-run nondeterminism in {key}"
    # resume from a saved state at step 12 continues bit-identically (Philox is counter-based)
    c = B.from_tiling(t, **p)
    c.step(12)
    sc = to_np(c.get_state())
    tt = w.Tiling(t.Lx, t.Ly, t.S, sc["pos"], sc["cell_vertex_num"], sc["cell_vertices"], sc["vertex_neighbors"],
                  sc["vertex_cell_neighbors"], sc["theta"])
    d = B.from_tiling(tt, **dict(p, step0=12))
    d.step(18)
    sd = to_np(d.get_state())
    for key in ("pos", "theta"):
        assert np.array_equal(sa[key], sd[key]), key
    h.assert_same_topology(sa, sd)


def test_host_pointer_entry_points_round_trip(B):
    t = tiling(1)
    p = w.config_params(1)
    gh = B.from_tiling(t, host=True, **p)
    gd = B.from_tiling(t, host=False, **p)
    gh.step(5)
    gd.step(5)
    sh = gh.get_state_host()
    sd = to_np(gd.get_state())
    for key in ("pos", "theta", "cell_vertices", "vertex_neighbors", "vertex_cell_neighbors", "cell_vertex_num"):
        assert np.array_equal(sh[key], sd[key]), key
    assert sh["stats"]["step"] == 5 and sh["stats"]["kernel_launches"] > 0


def test_create_rejects_inconsistent_topology(B):
    t = tiling(0).copy()
    t.vertex_cell_neighbors[5] = t.vertex_cell_neighbors[5][[1, 2, 0]]      # break the slot convention
    with pytest.raises(B.AvmError, match="inconsistent"):
        B.from_tiling(t, **w.config_params(0))
    t = tiling(0).copy()
    t.cell_vertex_num[3] = 17
    with pytest.raises(B.AvmError, match="inconsistent"):
        B.from_tiling(t, **w.config_params(0))
    t = tiling(0).copy()
    t.pos[0, 0] = np.nan
    with pytest.raises(B.AvmError, match="inconsistent"):
        B.from_tiling(t, **w.config_params(0))


def test_degenerate_cases(B):
    # l_c = 0: no T1 ever; Dr = 0, v0 = 0: pure gradient descent, energy decreases
    t = tiling(0)
    p = dict(w.config_params(0), l_c=0.0, v0=0.0, Dr=0.0, dt=1e-3)
    g = B.from_tiling(t, **p)
    E = [g.energy()]
    for _ in range(20):
        g.step(1)
        E.append(g.energy())
    assert all(b < a for a, b in zip(E, E[1:]))
    st = g.stats()
    assert st["t1_short"] == 0 and st["t1_flips"] == 0
    # pure activity: closed-form translation (same pin as the oracle's)
    th0 = 0.7
    hx = w.hex_tiling(6, 4, a=1.0, theta=np.full(24, th0))
    g = B.from_tiling(hx, KA=0.0, KP=0.0, v0=0.3, Dr=0.0, dt=0.01, l_c=0.0)
    g.step(250)
    s = to_np(g.get_state())
    expect = hx.pos + 250 * 0.3 * 0.01 * np.array([np.cos(th0), np.sin(th0)])
    assert_positions_close(s["pos"], expect, hx.Lx, hx.Ly, 1e-12)
    # zero steps is a no-op
    g.step(0)
    assert g.stats()["step"] == 250


def test_overflow_guard_on_gpu(B):
    t16 = tiling(1)
    nmax = int(t16.cell_vertex_num.max())
    assert nmax % 4 == 0, "cfg1's largest cell has 12 vertices"
    t = w.voronoi_tiling(4096, 64.0, 2, S=nmax)
    p = w.config_params(1)
    g = B.from_tiling(t, **p)
    o = oracle.from_tiling(t, **p)
    g.step(30)
    o.step(30)
    sg, so = to_np(g.get_state()), o.get_state()
    assert_states_match(sg, so, t.Lx, t.Ly)


@pytest.mark.parametrize("k,steps", [(3, 3), (4, 2)])
def test_full_size_configs_against_oracle(B, k, steps):
    """BASELINE.json's full sizes in the launch configuration bench.py times (Hilbert-sorted at
    create): whole-state comparison after a few steps, plus forces from the identical state."""
    t = tiling(k)
    p = w.config_params(k)
    g = B.from_tiling(t, **p)
    o = oracle.from_tiling(t, **p)
    F, ap = g.compute_forces()
    Fo, apo = o.compute_forces()
    assert_forces_close(F.cpu().numpy(), Fo, ap.cpu().numpy(), apo)
    del F, ap
    g.step(steps)
    o.step(steps)
    sg, so = to_np(g.get_state()), o.get_state()
    assert_states_match(sg, so, t.Lx, t.Ly)
    assert sg["stats"]["t1_flips"] > 1000
    L2 = t.Lx * t.Ly
    apg = g.compute_forces()[1].cpu().numpy()
    assert abs(apg[:, 0].sum() - L2) <= 1e-12 * L2
    # candidate and winner sets of the state both sides have reached, as sets of (tag_min, tag_max); the oracle's
    # state is loaded into a fresh simulation so that both decide from identical positions
    tt = w.Tiling(t.Lx, t.Ly, t.S, so["pos"], so["cell_vertex_num"], so["cell_vertices"], so["vertex_neighbors"],
                  so["vertex_cell_neighbors"], so["theta"])
    g.close()
    g2 = B.from_tiling(tt, **dict(p, step0=steps))
    cand, win = g2.debug_t1()
    co, wo = o.debug_t1()
    cg, wg = {tuple(x) for x in cand.tolist()}, {tuple(x) for x in win.tolist()}
    cs, ws = {tuple(x) for x in co.tolist()}, {tuple(x) for x in wo.tolist()}
    fuzzy = near_threshold(so, cg ^ cs, t.Lx, t.Ly, p["l_c"])
    assert (cg ^ cs) <= fuzzy
    assert len(cs) > 1000
    if not fuzzy:
        assert wg == ws
    g2.close()
    _TILINGS.pop(k, None)


def test_two_launch_schedule_equals_three_launch_schedule(B):
    """The default schedule applies the T1 flips of a step inside the next force/move launch
    (flagged vertices are moved after the flips); the plain schedule runs a third kernel per
    step.  Both must give the same bits, whatever the chunking of avm_step calls, including the
    step-0 burst (thousands of candidates: more candidates than flipper warps) and a re-sort."""
    t = tiling(1)
    p = dict(w.config_params(1), sort_every=7)
    keys = ("pos", "theta", "cell_vertices", "vertex_neighbors", "vertex_cell_neighbors", "cell_vertex_num")
    a = B.from_tiling(t, schedule="fused", **p)     # small systems default to the three-launch schedule
    a.step(40)
    sa = to_np(a.get_state())
    b = B.from_tiling(t, schedule="fused", **p)
    for n in (1, 1, 3, 5, 13, 17):
        b.step(n)
    sb = to_np(b.get_state())
    c = B.from_tiling(t, schedule="unfused", **p)
    c.step(40)
    sc = to_np(c.get_state())
    assert sa["stats"]["kernel_launches"] < sc["stats"]["kernel_launches"]
    for key in keys:
        assert np.array_equal(sa[key], sb[key]), f"chunking changes {key}: max diff {np.abs(sa[key] - sb[key]).max()}"
        assert np.array_equal(sa[key], sc[key]), \
            f"two-launch and three-launch schedules differ in {key}: max diff {np.abs(sa[key] - sc[key]).max()}"
    for key in ("t1_short", "t1_candidates", "t1_flips", "t1_blocked", "overflow_rejects", "error"):
        assert sa["stats"][key] == sb["stats"][key] == sc["stats"][key], key
    assert sa["stats"]["t1_flips"] > 100


def test_golden_trace_on_gpu(B):
    """the stored oracle trace of configs[0] (tests/golden/) reproduced by the CUDA path"""
    import json
    import os
    stored = json.load(open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "cfg0_oracle_trace.json")))
    t = tiling(0)
    g = B.from_tiling(t, **w.config_params(0))
    for r in stored["rows"]:
        g.step(r["step"] - g.stats()["step"])
        s = to_np(g.get_state())
        F, ap = g.compute_forces()
        ap = ap.cpu().numpy()
        assert s["stats"]["t1_flips"] == r["t1_flips"] and s["stats"]["t1_candidates"] == r["t1_candidates"]
        assert np.bincount(s["cell_vertex_num"], minlength=17).tolist() == r["cell_vertex_num_hist"]
        assert abs(ap[:, 0].sum() - r["sum_area"]) <= 1e-10 and abs(ap[:, 1].sum() - r["sum_perimeter"]) <= 1e-7
        assert abs(g.energy() - r["energy"]) <= 1e-7 * max(1.0, r["energy"])
        assert abs(s["theta"].sum() - r["theta_sum"]) <= 1e-8


@pytest.mark.parametrize("k,steps,sort_every", [(0, 100, 0), (1, 40, 9), (2, 6, 0)])
def test_repeated_t1_passes_match_the_oracle(B, k, steps, sort_every):
    """NEXT-1, the paper's own rule: T1 passes repeated within a step until none
    finds a candidate.  Topology and counters bit-exact, positions within the trajectory
    tolerance, and no candidate left after the last step."""
    t = tiling(k)
    p = dict(w.config_params(k), t1_max_passes=12)
    g = B.from_tiling(t, **dict(p, sort_every=sort_every))
    o = oracle.from_tiling(t, **p)
    one = oracle.from_tiling(t, **w.config_params(k))
    chunk = max(1, steps // 4)
    done = 0
    while done < steps:
        n = min(chunk, steps - done)
        g.step(n)
        o.step(n)
        done += n
        assert_states_match(to_np(g.get_state()), o.get_state(), t.Lx, t.Ly)
    one.step(steps)
    so = o.get_state()
    assert so["stats"]["t1_flips"] > 0
    if k > 0:   # blocked candidates flip within the same step: fewer candidates seen again later
        assert so["stats"]["t1_blocked"] != one.get_state()["stats"]["t1_blocked"] or \
            so["stats"]["t1_candidates"] != one.get_state()["stats"]["t1_candidates"]
    cand, _ = o.debug_t1()
    assert len(cand) == 0
    cg, wg = g.debug_t1()
    assert len(cg) == 0 and len(wg) == 0


def test_long_run_at_the_config_length_keeps_every_invariant(B):
    """configs[2] for its full 10^4 steps (fluid regime, ~60 flips per step, a re-sort every 500):
    far beyond what the oracle can follow, so what is checked is what holds at any length —
    a valid 3-coordinated tiling of the torus with the slot convention intact, areas tiling the
    box, a clean error word, and the create-validation accepting the exported state again."""
    t = tiling(2)
    p = dict(w.config_params(2), sort_every=500)
    g = B.from_tiling(t, **p)
    g.step(10000)
    s = to_np(g.get_state())
    assert s["stats"]["error"] == 0 and s["stats"]["n_sorts"] >= 20
    assert s["stats"]["t1_flips"] > 100000
    assert s["stats"]["t1_flips"] + s["stats"]["t1_blocked"] == s["stats"]["t1_candidates"]
    assert np.isfinite(s["pos"]).all() and (s["pos"] >= 0).all() and (s["pos"][:, 0] < t.Lx).all()
    h.check_topology(s["cell_vertex_num"], s["cell_vertices"], s["vertex_neighbors"], s["vertex_cell_neighbors"], S=t.S)
    ap = g.compute_forces()[1].cpu().numpy()
    L2 = t.Lx * t.Ly
    assert abs(ap[:, 0].sum() - L2) <= 1e-12 * L2
    assert (ap[:, 1] > 0).all()
    # the exported state is a consistent input (avm_create validates lists against each other)
    tt = w.Tiling(t.Lx, t.Ly, t.S, s["pos"], s["cell_vertex_num"], s["cell_vertices"], s["vertex_neighbors"],
                  s["vertex_cell_neighbors"], s["theta"])
    g2 = B.from_tiling(tt, **dict(p, step0=10000))
    g2.step(1)
    g.step(1)
    s1, s2 = to_np(g.get_state()), to_np(g2.get_state())
    assert np.array_equal(s1["pos"], s2["pos"]) and np.array_equal(s1["theta"], s2["theta"])


def test_two_launch_schedule_at_full_size_equals_three_launch_schedule(B):
    """configs[3] (N = 1,048,576, the bench workload) for 300 steps with a re-sort every 100, three ways:
    the two-launch schedule forced for every step (~96 000 simultaneous candidates in step 0: the
    many-candidate path inside force_move; later a few dozen per step: dedicated flipper warps),
    the schedule avm_step chooses by itself from the T1 load the device reports (stand-alone T1
    kernel during the burst, two launches afterwards), and the three-launch schedule.  Bit for bit."""
    t = tiling(3)
    p = dict(w.config_params(3), sort_every=100)
    keys = ("pos", "theta", "cell_vertices", "vertex_neighbors", "vertex_cell_neighbors", "cell_vertex_num")
    states = {}
    for name in ("fused", "auto", "unfused"):
        a = B.from_tiling(t, schedule=name, **p)
        if name == "auto":          # the host sees the reported load only as far as the device has come
            for n in (250, 50):
                a.step(n)
                a.stats()
        else:
            a.step(300)
        states[name] = to_np(a.get_state())
        if name == "fused":
            area = a.compute_forces()[1][:, 0].sum().item()
        a.close()
        del a
    sa, sb = states["fused"], states["unfused"]
    assert sa["stats"]["kernel_launches"] < states["auto"]["stats"]["kernel_launches"] < sb["stats"]["kernel_launches"]
    for other in ("auto", "unfused"):
        for key in keys:
            assert np.array_equal(sa[key], states[other][key]), (other, key)
        for key in ("t1_short", "t1_candidates", "t1_flips", "t1_blocked", "overflow_rejects", "error"):
            assert sa["stats"][key] == states[other]["stats"][key], (other, key)
    assert sa["stats"]["error"] == 0 and sa["stats"]["t1_flips"] > 90000
    L2 = t.Lx * t.Ly
    assert abs(area - L2) <= 1e-12 * L2
    _TILINGS.pop(3, None)


@pytest.mark.parametrize("k,steps", [(0, 25), (1, 10)])
def test_observables_match_the_oracle(B, k, steps):
    """NEXT-2: avm_observe against the numpy definitions on the oracle's geometry, on the start
    tiling and inside the step-0 burst (where some cells are transiently inverted)."""
    t = tiling(k)
    p = w.config_params(k)
    g = B.from_tiling(t, **dict(p, sort_at_create=True))
    o = oracle.from_tiling(t, **p)
    for n in (0, 1, steps):
        g.step(n)
        o.step(n)
        a, b = g.observe(), o.observables()
        for key in ("energy", "sum_area", "sum_perimeter", "mean_shape_index", "area_min", "area_max", "area_variance"):
            assert abs(a[key] - b[key]) <= 1e-9 * max(1.0, abs(b[key])), (n, key, a[key], b[key])
        assert a["n_nonpositive_area"] == b["n_nonpositive_area"]
        assert a["step"] == o.get_state()["stats"]["step"] and a["t1_flips"] == o.get_state()["stats"]["t1_flips"]
        assert abs(a["energy"] - g.energy()) == 0.0
    assert abs(a["sum_area"] - t.Lx * t.Ly) <= 1e-12 * t.Lx * t.Ly


@pytest.mark.parametrize("k,steps,sort_every", [(0, 60, 0), (1, 24, 7)])
def test_per_cell_targets_match_the_oracle(B, k, steps, sort_every):
    """NEXT-4: per-cell preferred area and perimeter of Eq. 1 (a bidisperse mixture): forces within
    1e-10, trajectory within 1e-8 with bit-exact topology (re-sorts included), energy, and
    NULL, NULL restoring the uniform path."""
    t = tiling(k)
    p = w.config_params(k)
    rng = np.random.default_rng(11)
    big = rng.random(t.N) < 0.5
    A0 = np.where(big, 1.25, 0.75)
    P0 = np.where(big, 3.9 * np.sqrt(1.25), 3.7 * np.sqrt(0.75))
    g = B.from_tiling(t, **dict(p, sort_every=sort_every, sort_at_create=True))
    o = oracle.from_tiling(t, **p)
    g.set_cell_targets(A0, P0)
    o.set_cell_targets(A0, P0)
    F, ap = g.compute_forces()
    Fo, apo = o.compute_forces()
    assert_forces_close(F.cpu().numpy(), Fo, ap.cpu().numpy(), apo)
    assert abs(g.energy() - o.energy()) <= 1e-10 * abs(o.energy())
    g.step(steps)
    o.step(steps)
    assert_states_match(to_np(g.get_state()), o.get_state(), t.Lx, t.Ly)
    assert abs(g.energy() - o.energy()) <= 1e-8 * abs(o.energy())
    uni = oracle.from_tiling(t, **p)
    uni.step(steps)
    assert np.abs(uni.get_state()["pos"] - o.get_state()["pos"]).max() > 1e-3      # the targets matter
    g.set_cell_targets(None, None)
    o.set_cell_targets(None, None)
    F, ap = g.compute_forces()
    Fo, apo = o.compute_forces()
    assert_forces_close(F.cpu().numpy(), Fo, ap.cpu().numpy(), apo)


@pytest.mark.parametrize("S", [20, 32])
@pytest.mark.parametrize("fused", [False, True])
def test_other_row_strides_match_the_oracle(B, S, fused):
    """rows longer than 16 entries use different code (one row per pass in the flippers, planes
    4..7 of the padded rows, bit 31 of the short-edge mask): configs[1] geometry with S = 20 and
    the maximum S = 32, in both schedules, through the step-0 burst."""
    t = w.voronoi_tiling(4096, 64.0, 2, S=S)
    p = dict(w.config_params(1), schedule="fused" if fused else "unfused")
    g = B.from_tiling(t, **dict(p, sort_every=6, sort_at_create=True))
    o = oracle.from_tiling(t, **p)
    F, ap = g.compute_forces()
    Fo, apo = o.compute_forces()
    assert_forces_close(F.cpu().numpy(), Fo, ap.cpu().numpy(), apo)
    g.step(25)
    o.step(25)
    assert_states_match(to_np(g.get_state()), o.get_state(), t.Lx, t.Ly)
    assert o.get_state()["stats"]["t1_flips"] > 300


def test_smallest_tori(B):
    """the smallest tilings the generator builds with valid minimum-image unwrapping (3 x 4 and
    4 x 4 hexagons: N = 12 and 16, a single CTA, more flipper warps than candidates), many steps
    with strong activity and a large threshold so that flips keep happening (22 and 59 flips, blocked
    candidates included); positions to 1e-8 (the band excluded from the comparison of T1 decisions is 1e-9 wide:
    a flip decided differently would show up as a topology mismatch)"""
    for nx, ny in ((3, 4), (4, 4)):
        t = w.hex_tiling(nx, ny, a=1.0)
        p = dict(KA=1.0, KP=1.0, A0=2.0, P0=6.5, v0=1.0, Dr=1.0, dt=0.01, l_c=0.6, seed=3)
        g = B.from_tiling(t, **p)
        o = oracle.from_tiling(t, **p)
        for _ in range(4):
            g.step(50)
            o.step(50)
            assert_states_match(to_np(g.get_state()), o.get_state(), t.Lx, t.Ly, pos_tol=1e-8)
        assert o.get_state()["stats"]["t1_flips"] >= 20


@pytest.mark.parametrize("params_of", [3, 4])
def test_fused_schedule_hammered_at_a_million_cells(B, params_of):
    """The two-launch schedule against the three-launch schedule over 2000 steps with re-sorts on the
    N = 1,048,576 tiling, bit for bit: with configs[3]'s parameters (after the burst a few dozen
    candidates per step: dedicated flipper warps work while every other warp sweeps, the regime
    in which a skipped vertex must stay skipped for the whole launch) and with configs[4]'s
    parameters (thousands of candidates in every step: the many-candidate path).  The flagged-vertex
    bitmap is read-only for the launch that sweeps with it, so both are race-free by construction;
    this test is the empirical side of that argument (compute-sanitizer is closed on this pool)."""
    t = tiling(3)
    p = dict(w.config_params(3), sort_every=250)
    if params_of == 4:
        p4 = w.config_params(4)
        p.update({k: p4[k] for k in ("P0", "v0", "Dr", "dt", "l_c")})
    keys = ("pos", "theta", "cell_vertices", "vertex_neighbors", "vertex_cell_neighbors", "cell_vertex_num")
    out = []
    for sched in ("fused", "unfused", "fused"):
        a = B.from_tiling(t, schedule=sched, **p)
        a.step(2000)
        out.append(to_np(a.get_state()))
        a.close()
        del a
    for other in out[1:]:
        for key in keys:
            assert np.array_equal(out[0][key], other[key]), key
        for key in ("t1_short", "t1_candidates", "t1_flips", "t1_blocked", "overflow_rejects", "error"):
            assert out[0]["stats"][key] == other["stats"][key], key
    assert out[0]["stats"]["error"] == 0 and out[0]["stats"]["n_sorts"] == 9      # one at create, eight in the run
    assert out[0]["stats"]["t1_flips"] > (2_000_000 if params_of == 4 else 100_000)
    _TILINGS.pop(3, None)


def test_fused_schedule_with_resorts_against_the_oracle_at_fused_size(B):
    """configs[4]'s parameters and density on the smallest tiling that takes the two-launch schedule by
    default (V = 2^20), re-sorted every 3 steps, followed by the oracle across two re-sort
    boundaries: pending flips are completed before each re-sort, the candidate lists hold pre-sort
    indices and are dropped, tags keep priorities and noise unchanged (R11, R16)."""
    N = 524288
    cfg = w.CONFIGS[4]
    L = cfg["L"] * (N / cfg["N"]) ** 0.5
    t = w.voronoi_tiling(N, L, cfg["points_seed"])
    p = dict(w.config_params(4), Lx=L, Ly=L, sort_every=3, sort_at_create=True)
    o = oracle.from_tiling(t, **p)
    for sched in ("fused", "auto"):
        g = B.from_tiling(t, schedule=sched, **p)
        if sched == "fused":
            g.step(7)
            o.step(7)
        else:
            g.step(4)
            g.step(3)
        sg = to_np(g.get_state())
        assert_states_match(sg, o.get_state(), t.Lx, t.Ly)
        assert sg["stats"]["n_sorts"] == 3 and sg["stats"]["t1_flips"] > 10000
        g.close()


def test_sub_step_order_on_gpu(B):
    """GPU twins of the oracle's R7 / R6 pins: the move uses the directors of the start of the step
    (closed form with Dr > 0), and an edge brought below l_c by the move flips in that very step."""
    t = tiling(0)
    v0, dt, Dr, seed = 0.7, 0.01, 2.0, 11
    g = B.from_tiling(t, KA=0.0, KP=0.0, v0=v0, Dr=Dr, dt=dt, l_c=0.0, seed=seed)
    th1 = t.theta + np.sqrt(2 * Dr * dt) * oracle.director_noise(seed, 0, 0, t.N)

    def drift(th):
        n = np.stack([np.cos(th), np.sin(th)], axis=1)
        return dt * v0 / 3.0 * n[t.vertex_cell_neighbors].sum(axis=1)
    g.step(1)
    s1 = to_np(g.get_state())
    assert_positions_close(s1["pos"], np.mod(t.pos + drift(t.theta), [t.Lx, t.Ly]), t.Lx, t.Ly, 1e-14)
    assert np.abs(s1["theta"] - th1).max() < 1e-14
    g.step(1)
    s2 = to_np(g.get_state())
    assert_positions_close(s2["pos"], np.mod(s1["pos"] + drift(s1["theta"]), [t.Lx, t.Ly]), t.Lx, t.Ly, 1e-14)
    # R6: same construction as tests/test_oracle_integrator.py
    from tests.test_oracle_t1 import edge_cells_from_rows, shrink_edge
    l_c, dt, v0 = 0.04, 0.01, 0.9
    hx = w.hex_tiling(6, 4, a=1.0)
    v1 = 7
    v2 = int(hx.vertex_neighbors[v1, 1])
    lo, hi = min(v1, v2), max(v1, v2)
    L, R, E1, E2 = edge_cells_from_rows(hx.cell_vertex_num, hx.cell_vertices, hx.vertex_cell_neighbors, lo, hi)
    closing = dt * 2.0 * v0 / 3.0
    pos, m, u = shrink_edge(hx, lo, hi, l_c + 0.5 * closing)
    theta = np.zeros(hx.N)
    theta[E1], theta[E2] = np.arctan2(u[1], u[0]), np.arctan2(-u[1], -u[0])
    theta[L] = theta[R] = 0.3
    tt = w.Tiling(hx.Lx, hx.Ly, hx.S, pos, hx.cell_vertex_num, hx.cell_vertices, hx.vertex_neighbors,
                  hx.vertex_cell_neighbors, theta)
    for sched in ("fused", "unfused"):
        g = B.from_tiling(tt, KA=0.0, KP=0.0, v0=v0, Dr=0.0, dt=dt, l_c=l_c, schedule=sched)
        cand, _ = g.debug_t1()
        assert len(cand) == 0
        g.step(1)
        s = to_np(g.get_state())
        assert s["stats"]["t1_short"] == 1 and s["stats"]["t1_flips"] == 1
        assert h.cells_adjacent(s["cell_vertices"], s["cell_vertex_num"], E1, E2)


def test_repeated_passes_overflow_on_a_later_pass(B):
    """GPU twin of the oracle pin: t1_short / overflow_rejects are first-pass statistics, the sticky
    error bit 2 is raised by whichever pass first sees the overflow (local re-detection included)."""
    from tests.test_oracle_t1 import overflow_on_a_later_pass_case
    tt, kw, E, _ = overflow_on_a_later_pass_case()
    for passes in (4, 1):
        g = B.from_tiling(tt, t1_max_passes=passes, **kw)
        o = oracle.from_tiling(tt, t1_max_passes=passes, **kw)
        for _ in range(2):
            g.step(1)
            o.step(1)
            assert_states_match(to_np(g.get_state()), o.get_state(), tt.Lx, tt.Ly)
        assert o.get_state()["stats"]["error"] == 2


@pytest.mark.parametrize("k,steps,sort_every", [(0, 60, 0), (1, 24, 7)])
def test_per_cell_moduli_match_the_oracle(B, k, steps, sort_every):
    """NEXT-4: per-cell K_A,i, K_P,i together with per-cell targets (Eq. 1): forces within 1e-10,
    trajectory within 1e-8 with bit-exact topology (re-sorts included), energy; each pair can be
    switched back to the uniform values independently."""
    t = tiling(k)
    p = w.config_params(k)
    rng = np.random.default_rng(12)
    soft = rng.random(t.N) < 0.5
    KA, KP = np.where(soft, 0.4, 1.7), np.where(soft, 0.6, 1.2)
    A0, P0 = np.where(soft, 1.2, 0.8), np.where(soft, 3.9 * np.sqrt(1.2), 3.7 * np.sqrt(0.8))
    g = B.from_tiling(t, **dict(p, sort_every=sort_every, sort_at_create=True))
    o = oracle.from_tiling(t, **p)
    g.set_cell_moduli(KA, KP)
    o.set_cell_moduli(KA, KP)
    F, ap = g.compute_forces()
    Fo, apo = o.compute_forces()
    assert_forces_close(F.cpu().numpy(), Fo, ap.cpu().numpy(), apo)
    g.set_cell_targets(A0, P0)
    o.set_cell_targets(A0, P0)
    F, ap = g.compute_forces()
    Fo, apo = o.compute_forces()
    assert_forces_close(F.cpu().numpy(), Fo, ap.cpu().numpy(), apo)
    assert abs(g.energy() - o.energy()) <= 1e-10 * abs(o.energy())
    g.step(steps)
    o.step(steps)
    assert_states_match(to_np(g.get_state()), o.get_state(), t.Lx, t.Ly)
    assert abs(g.energy() - o.energy()) <= 1e-8 * abs(o.energy())
    assert o.get_state()["stats"]["t1_flips"] > 0
    g.set_cell_targets(None, None)           # moduli stay heterogeneous
    o.set_cell_targets(None, None)
    F, ap = g.compute_forces()
    Fo, apo = o.compute_forces()
    assert_forces_close(F.cpu().numpy(), Fo, ap.cpu().numpy(), apo)
    g.set_cell_moduli(None, None)
    o.set_cell_moduli(None, None)
    F, ap = g.compute_forces()
    Fo, apo = o.compute_forces()
    assert_forces_close(F.cpu().numpy(), Fo, ap.cpu().numpy(), apo)
    g.step(5)
    o.step(5)
    assert_states_match(to_np(g.get_state()), o.get_state(), t.Lx, t.Ly)


@pytest.mark.parametrize("sched", ["fused", "unfused"])
def test_mean_square_displacement_matches_the_oracle(B, sched):
    """NEXT-2: MSD from the image counts the library keeps (vertices leave through the box boundary, T1s
    reposition their end points, the Hilbert re-sort permutes everything) against the oracle's
    unwrapped positions; closed-form pure-activity translation; reset."""
    t = tiling(0)
    p = dict(w.config_params(0), v0=3.0, Dr=0.2, sort_every=11, sort_at_create=True, schedule=sched)
    g = B.from_tiling(t, **p)
    o = oracle.from_tiling(t, **p)
    assert g.observe()["msd"] == 0.0
    for n in (1, 9, 90, 200):
        g.step(n)
        o.step(n)
        a, b = g.observe()["msd"], o.msd()
        assert abs(a - b) <= 1e-9 * max(b, 1e-12), (n, a, b)
    assert o.get_state()["stats"]["t1_flips"] > 0 and b > 0.5
    g.msd_reset()
    o.msd_reset()
    assert g.observe()["msd"] == 0.0
    g.step(30)
    o.step(30)
    assert abs(g.observe()["msd"] - o.msd()) <= 1e-9 * o.msd()
    th0 = 2.1
    hx = w.hex_tiling(6, 4, a=1.0, theta=np.full(24, th0))
    g = B.from_tiling(hx, KA=0.0, KP=0.0, v0=0.8, Dr=0.0, dt=0.01, l_c=0.0, schedule=sched)
    g.step(1500)
    assert abs(g.observe()["msd"] - 144.0) < 1e-9 * 144.0


@pytest.mark.parametrize("seed", [4, 1])
def test_image_counts_are_applied_once_when_movers_overlap(B, seed):
    """in the two-launch schedule the post-flip movers run once per T1 candidate, so a vertex of a cell
    that two candidates touch (or met again in a later pass over a long row) is moved more than once in a step.
    The move is idempotent, the image count of the mean-square displacement is an increment: it must be applied
    once.  The tiling translates rigidly (no forces, one common director) by a fifth of the box per step, so a
    third of the vertices cross the boundary in every step and the MSD is (n v0 dt)^2 up to the end points that T1s
    reposition; a vertex counted twice adds 64^2 / 8192 = 0.5.  (The library that incremented per mover gave
    4101.8 and 4102.6 instead of 4096.0 on these two tilings.)  The steps must come in ONE call: the last step of
    a call always completes with the stand-alone T1 kernel.  Exact equality with the three-launch schedule, and
    the oracle's unwrapped positions."""
    t = w.voronoi_tiling(4096, 64.0, seed)
    t.theta[:] = 0.6
    p = dict(KA=0.0, KP=0.0, A0=1.0, P0=3.8, v0=128.0, Dr=0.0, mu=1.0, dt=0.1, l_c=0.008, seed=11)
    f = B.from_tiling(t, schedule="fused", **p)
    u = B.from_tiling(t, schedule="unfused", **p)
    o = oracle.from_tiling(t, **p)
    for n in (5, 10):
        f.step(5)
        u.step(5)
        o.step(5)
        a = f.observe()["msd"]
        assert a == u.observe()["msd"], (n, a, u.observe()["msd"])
        assert abs(a - o.msd()) <= 1e-9 * o.msd()
        assert abs(a - (12.8 * n) ** 2) < 1e-3
    sf, su = f.stats(), u.stats()
    assert sf["kernel_launches"] < su["kernel_launches"] - 6                    # it really ran two launches per step
    assert 20 < sf["t1_candidates"] <= 85 and sf["t1_blocked"] > 0               # one warp per candidate, with shared cells
    assert np.array_equal(to_np(f.get_state())["pos"], to_np(u.get_state())["pos"])


@pytest.mark.parametrize("k,steps,sort_every", [(0, 150, 0), (1, 60, 7), (2, 20, 6)])
def test_persistent_schedule_equals_the_launched_schedules(B, k, steps, sort_every):
    """Launch-free stepping (one cooperative launch per call / per stretch between re-sorts, grid-wide
    barriers between the stages) against one launch per kernel, bit for bit and for any chunking;
    configs[0] runs as a single CTA, configs[2] with more work than resident threads."""
    t = tiling(k)
    p = dict(w.config_params(k), sort_every=sort_every)
    keys = ("pos", "theta", "cell_vertices", "vertex_neighbors", "vertex_cell_neighbors", "cell_vertex_num")
    a = B.from_tiling(t, schedule="persistent", **p)
    a.step(steps)
    sa = to_np(a.get_state())
    b = B.from_tiling(t, schedule="persistent", **p)
    for n in (1, 2, steps - 3):
        b.step(n)
    sb = to_np(b.get_state())
    c = B.from_tiling(t, schedule="unfused", **p)
    c.step(steps)
    sc = to_np(c.get_state())
    assert sa["stats"]["kernel_launches"] < sc["stats"]["kernel_launches"] - 2 * steps     # re-sorts are launched in both
    for other in (sb, sc):
        for key in keys:
            assert np.array_equal(sa[key], other[key]), key
        for key in ("t1_short", "t1_candidates", "t1_flips", "t1_blocked", "overflow_rejects", "error", "n_sorts"):
            assert sa["stats"][key] == other["stats"][key], key
    assert sa["stats"]["t1_flips"] > 0
    assert abs(a.observe()["msd"] - c.observe()["msd"]) == 0.0


@pytest.mark.parametrize("k,steps,sort_every", [(0, 7, 0), (1, 5, 3), (2, 4, 0)])
def test_observing_geometry_pass_matches_the_oracle(B, k, steps, sort_every):
    """NEXT-2, reductions fused into the geometry pass: avm_step_observe reduces the observables of the
    moved tiling of its last step (after the move and the director update, before the T1 pass) inside
    the cell pass.  Oracle side: the same step taken in its two halves, the numpy definitions evaluated
    in between.  The step itself is unchanged: states match afterwards, and a further plain step too."""
    t = w.config_tiling(k)
    p = w.config_params(k)
    g = B.from_tiling(t, **dict(p, sort_every=sort_every, sort_at_create=sort_every > 0))
    o = oracle.from_tiling(t, **p)
    for rep in range(3):
        og = g.step_observe(steps)
        o.step(steps - 1)
        o.step_move_and_rotate()
        oo = o.observables()
        o.step_topology_and_advance()
        for key in ("energy", "sum_area", "sum_perimeter", "mean_shape_index", "area_min", "area_max", "area_variance", "msd"):
            assert abs(og[key] - oo[key]) <= 1e-9 * max(1.0, abs(oo[key])), (rep, key, og[key], oo[key])
        assert og["n_nonpositive_area"] == oo["n_nonpositive_area"]
        so = o.get_state()
        assert og["step"] == so["stats"]["step"] and og["t1_flips"] == so["stats"]["t1_flips"]
        assert_states_match(to_np(g.get_state()), so, t.Lx, t.Ly)
    assert so["stats"]["t1_flips"] > 0 or k == 0
    # observing costs nothing afterwards: the between-steps observables agree too
    a, b = g.observe(), o.observables()
    assert abs(a["energy"] - b["energy"]) <= 1e-9 * abs(b["energy"]) and abs(a["msd"] - b["msd"]) <= 1e-9 * max(1.0, b["msd"])


@pytest.mark.parametrize("N,L", [(300, 17.3), (1500, 38.7), (4000, 63.2)])
def test_cluster_persistent_default_at_ragged_sizes(B, N, L):
    """Systems of 513..8192 vertices step by default inside one thread-block cluster (hardware cluster barrier,
    two vertices per thread and trip).  Sizes that fill the last CTA only partly, per-cell parameters, a re-sort
    period that cuts the call into stretches: the default must equal one launch per kernel bit for bit and follow
    the oracle."""
    t = w.voronoi_tiling(N, L, 31 + N)
    p = dict(KA=1.0, KP=1.0, A0=1.0, P0=3.9, v0=0.4, Dr=1.0, mu=1.0, dt=0.01, l_c=0.08, seed=5, sort_every=9)
    rng = np.random.default_rng(N)
    A0 = 1.0 + 0.2 * rng.standard_normal(N)
    P0 = 3.9 + 0.1 * rng.standard_normal(N)
    a = B.from_tiling(t, **p)                       # default: persistent, one cluster
    c = B.from_tiling(t, schedule="unfused", **p)
    o = oracle.from_tiling(t, **{k: v for k, v in p.items() if k != "sort_every"})
    for sim in (a, c, o):
        sim.set_cell_targets(A0, P0)
    for n in (1, 17, 40):
        a.step(n)
        c.step(n)
        o.step(n)
    sa, sc = to_np(a.get_state()), to_np(c.get_state())
    assert sa["stats"]["kernel_launches"] < sc["stats"]["kernel_launches"] - 100
    for key in ("pos", "theta", "cell_vertices", "vertex_neighbors", "vertex_cell_neighbors", "cell_vertex_num"):
        assert np.array_equal(sa[key], sc[key]), key
    assert sa["stats"]["t1_flips"] == sc["stats"]["t1_flips"] > 20
    assert_states_match(sa, o.get_state(), t.Lx, t.Ly)
