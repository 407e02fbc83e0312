"""Pins for the oracle's T1 pass (Fig. 1 right :27; R9-R12).

Hand-built neighbour exchange on a hexagonal torus, topological invariants after every pass of a
real trajectory, and a brute-force restatement of the candidate and conflict rules in Python
that derives the four cells of an edge from the cell ROWS (not from the slot convention)."""
import numpy as np
import pytest

import oracle
from paper_1702_02939_b200 import workloads as w
from tests import helpers as h


def edge_cells_from_rows(cvn, cv, vc, v, wv):
    """(L, R, E1, E2) of directed edge v->wv from the rows alone: L has (v, wv) consecutive in its
    CCW row, R has (wv, v); E1 / E2 are the remaining cells of v / wv."""
    L = R = None
    for c in vc[v]:
        row = cv[c, :cvn[c]].tolist()
        j = row.index(v)
        if row[(j + 1) % len(row)] == wv:
            L = c
        if row[(j - 1) % len(row)] == wv:
            R = c
    E1 = [c for c in vc[v] if c not in (L, R)]
    E2 = [c for c in vc[wv] if c not in (L, R)]
    assert L is not None and R is not None and len(E1) == 1 and len(E2) == 1
    return int(L), int(R), int(E1[0]), int(E2[0])


def brute_force_t1(state, Lx, Ly, l_c, S):
    """Candidates (R9, R10) and winners (R11) by exhaustive search."""
    pos, cvn, cv = state["pos"], state["cell_vertex_num"], state["cell_vertices"]
    vn, vc = state["vertex_neighbors"], state["vertex_cell_neighbors"]
    cands = []
    for v in range(pos.shape[0]):
        for wv in vn[v]:
            if not v < wv:
                continue
            d = pos[wv] - pos[v]
            l = np.hypot(h.min_image(d[0], Lx), h.min_image(d[1], Ly))
            if not l < l_c:
                continue
            L, R, E1, E2 = edge_cells_from_rows(cvn, cv, vc, v, int(wv))
            if len({L, R, E1, E2}) != 4:
                continue
            if not (cvn[L] > 3 and cvn[R] > 3 and cvn[E1] < S and cvn[E2] < S):
                continue
            cands.append(((v, int(wv)), {L, R, E1, E2}))
    winners = []
    for key, cells in cands:
        blocked = any(k2 < key and (cells & c2) for k2, c2 in cands)
        if not blocked:
            winners.append(key)
    return sorted(k for k, _ in cands), sorted(winners)


def shrink_edge(t, v1, v2, new_len):
    pos = t.pos.copy()
    d = pos[v2] - pos[v1]
    d = np.array([h.min_image(d[0], t.Lx), h.min_image(d[1], t.Ly)])
    m = pos[v1] + 0.5 * d
    u = d / np.linalg.norm(d)
    pos[v1] = np.mod(m - 0.5 * new_len * u, [t.Lx, t.Ly])
    pos[v2] = np.mod(m + 0.5 * new_len * u, [t.Lx, t.Ly])
    return pos, m, u


@pytest.mark.parametrize("v1,slot", [(7, 0), (7, 1), (7, 2), (20, 1)])
def test_hand_built_t1_exchanges_neighbours(v1, slot):
    """Fig. 1 (right): cells i,k adjacent before, cells j,l adjacent after; the edge is rotated by
    +90 degrees about its midpoint to length 1.5 l_c (R9)."""
    l_c = 0.04
    t = w.hex_tiling(6, 4, a=1.0)
    v2 = int(t.vertex_neighbors[v1, slot])
    lo, hi = min(v1, v2), max(v1, v2)
    pos, m, u = shrink_edge(t, lo, hi, 0.5 * l_c)
    L, R, E1, E2 = edge_cells_from_rows(t.cell_vertex_num, t.cell_vertices, t.vertex_cell_neighbors, lo, hi)
    assert h.cells_adjacent(t.cell_vertices, t.cell_vertex_num, L, R)
    assert not h.cells_adjacent(t.cell_vertices, t.cell_vertex_num, E1, E2)
    sim = oracle.from_tiling(t, l_c=l_c)
    sim.set_positions(pos)
    cand, win = sim.debug_t1()
    assert cand.tolist() == [[lo, hi]] and win.tolist() == [[lo, hi]]
    sim.t1_pass()
    s = sim.get_state()
    cvn, cv, vn, vc = s["cell_vertex_num"], s["cell_vertices"], s["vertex_neighbors"], s["vertex_cell_neighbors"]
    h.check_topology(cvn, cv, vn, vc)
    assert not h.cells_adjacent(cv, cvn, L, R)          # i,k no longer adjacent
    assert h.cells_adjacent(cv, cvn, E1, E2)            # j,l adjacent now
    assert cvn[L] == 5 and cvn[R] == 5 and cvn[E1] == 7 and cvn[E2] == 7
    assert s["stats"]["t1_flips"] == 1 and s["stats"]["t1_candidates"] == 1 and s["stats"]["t1_blocked"] == 0
    # which vertex went where: lo stays in R and joins both end cells, hi stays in L
    assert lo in cv[R] and lo not in cv[L] and hi in cv[L] and hi not in cv[R]
    assert lo in cv[E1] and lo in cv[E2] and hi in cv[E1] and hi in cv[E2]
    # geometry: midpoint kept, new edge = old direction rotated by +90 degrees, length 1.5 l_c
    d = s["pos"][hi] - s["pos"][lo]
    d = np.array([h.min_image(d[0], t.Lx), h.min_image(d[1], t.Ly)])
    assert abs(np.linalg.norm(d) - 1.5 * l_c) < 1e-14
    rot = np.array([-u[1], u[0]])
    assert np.allclose(d / np.linalg.norm(d), rot, atol=1e-12)
    mid = s["pos"][lo] + 0.5 * d
    dm = mid - m
    assert abs(h.min_image(dm[0], t.Lx)) < 1e-13 and abs(h.min_image(dm[1], t.Ly)) < 1e-13
    # rows stay counter-clockwise and still tile the box
    ap = h.polygon_areas_numpy(s["pos"], cvn, cv, t.Lx, t.Ly)
    assert (ap[:, 0] > 0).all()
    assert abs(ap[:, 0].sum() - t.Lx * t.Ly) < 1e-12 * t.Lx * t.Ly
    # everything not in the closure of the four cells is untouched
    touched = set(cv[[L, R, E1, E2]].ravel().tolist()) - {-1}
    others = np.array(sorted(set(range(t.V)) - touched))
    assert np.array_equal(vn[others], t.vertex_neighbors[others])
    assert np.array_equal(vc[others], t.vertex_cell_neighbors[others])
    assert np.array_equal(s["pos"][others], pos[others])


def test_flipping_back_restores_adjacency():
    """Two successive T1s on the same edge return the original cell adjacency (the second flip
    exchanges j,l back to i,k)."""
    l_c = 0.04
    t = w.hex_tiling(6, 4, a=1.0)
    v1, v2 = 7, int(t.vertex_neighbors[7, 0])
    lo, hi = min(v1, v2), max(v1, v2)
    pos, _, _ = shrink_edge(t, lo, hi, 0.5 * l_c)
    L, R, E1, E2 = edge_cells_from_rows(t.cell_vertex_num, t.cell_vertices, t.vertex_cell_neighbors, lo, hi)
    sim = oracle.from_tiling(t, l_c=l_c)
    sim.set_positions(pos)
    sim.t1_pass()
    s = sim.get_state()
    # shrink the new edge again and flip once more
    t2 = t.copy()
    t2.pos = s["pos"]
    pos2, _, _ = shrink_edge(t2, lo, hi, 0.5 * l_c)
    sim.set_positions(pos2)
    sim.t1_pass()
    s2 = sim.get_state()
    cvn, cv = s2["cell_vertex_num"], s2["cell_vertices"]
    h.check_topology(cvn, cv, s2["vertex_neighbors"], s2["vertex_cell_neighbors"])
    assert h.cells_adjacent(cv, cvn, L, R) and not h.cells_adjacent(cv, cvn, E1, E2)
    assert (cvn == 6).all()


def test_conflict_chain_only_smallest_key_flips():
    """R11: in a chain e1 < e2 < e3 of candidates sharing cells pairwise only e1 flips, because a
    candidate is blocked by any smaller candidate, not only by a winner."""
    l_c = 0.04
    t = w.hex_tiling(8, 6, a=1.0)
    # three consecutive edges along a zig-zag path of one cell's boundary share that cell
    c = 20
    row = t.cell_vertices[c, :6]
    pos = t.pos.copy()
    edges = [(int(row[0]), int(row[1])), (int(row[2]), int(row[3])), (int(row[4]), int(row[5]))]
    tt = t.copy()
    for a, b in edges:
        tt.pos = pos
        pos, _, _ = shrink_edge(tt, min(a, b), max(a, b), 0.5 * l_c)
    sim = oracle.from_tiling(t, l_c=l_c)
    sim.set_positions(pos)
    cand, win = sim.debug_t1()
    keys = sorted((min(a, b), max(a, b)) for a, b in edges)
    assert [tuple(x) for x in cand.tolist()] == keys
    assert [tuple(x) for x in win.tolist()] == [keys[0]]
    sim.t1_pass()
    st = sim.get_state()["stats"]
    assert st["t1_flips"] == 1 and st["t1_blocked"] == 2 and st["t1_candidates"] == 3


def test_triangle_guard_and_overflow_guard():
    """R10: a short edge on a triangle is not a candidate (it would create a 2-gon), and a short
    edge whose end cell is already at the stride is counted as an overflow reject."""
    t = w.voronoi_tiling(4096, 64.0, 2)
    tri = np.where(t.cell_vertex_num == 3)[0]
    assert len(tri) > 0
    c = int(tri[0])
    a, b = int(t.cell_vertices[c, 0]), int(t.cell_vertices[c, 1])
    pos, _, _ = shrink_edge(t, min(a, b), max(a, b), 1e-3)
    sim = oracle.from_tiling(t, l_c=2e-3)
    sim.set_positions(pos)
    cand, win = sim.debug_t1()
    assert [min(a, b), max(a, b)] not in cand.tolist()
    # overflow: rebuild the same tiling with stride = its largest cell; pick an edge ending on it
    nmax = int(t.cell_vertex_num.max())
    t8 = w.voronoi_tiling(4096, 64.0, 2, S=nmax)
    big = int(np.argmax(t8.cell_vertex_num))
    found = None
    for v in t8.cell_vertices[big, :nmax]:
        for k in range(3):
            wv = int(t8.vertex_neighbors[v, k])
            L, R, E1, E2 = edge_cells_from_rows(t8.cell_vertex_num, t8.cell_vertices, t8.vertex_cell_neighbors, int(v), wv)
            if E1 == big and t8.cell_vertex_num[L] > 3 and t8.cell_vertex_num[R] > 3 and len({L, R, E1, E2}) == 4:
                found = (int(v), wv)
    assert found is not None
    a, b = found
    pos, _, _ = shrink_edge(t8, min(a, b), max(a, b), 1e-4)
    sim = oracle.from_tiling(t8, l_c=2e-4)
    sim.set_positions(pos)
    cand, _ = sim.debug_t1()
    assert [min(a, b), max(a, b)] not in cand.tolist()
    sim.t1_pass()
    st = sim.get_state()["stats"]
    assert st["overflow_rejects"] == 1 and st["error"] & 2
    # with room in the rows (stride 16) the very same edge is a candidate
    sim16 = oracle.from_tiling(t, l_c=2e-4)
    sim16.set_positions(pos)
    cand16, _ = sim16.debug_t1()
    assert [min(a, b), max(a, b)] in cand16.tolist()
    sim16.t1_pass()
    assert sim16.get_state()["stats"]["overflow_rejects"] == 0


@pytest.mark.parametrize("k,steps", [(0, 100)])
def test_trajectory_invariants_and_bruteforce_rule(k, steps):
    """configs[0] for 100 steps: after every step the tiling is still a valid 3-coordinated
    torus, areas tile the box, and the candidate/winner sets equal the brute-force rule."""
    t = w.config_tiling(k)
    p = w.config_params(k)
    sim = oracle.from_tiling(t, **p)
    L2 = t.Lx * t.Ly
    total_flips = 0
    for s_i in range(steps):
        sim.step(1)
        s = sim.get_state()
        h.check_topology(s["cell_vertex_num"], s["cell_vertices"], s["vertex_neighbors"], s["vertex_cell_neighbors"])
        ap = sim.geometry()
        assert abs(ap[:, 0].sum() - L2) <= 1e-12 * L2
        ref = h.polygon_areas_numpy(s["pos"], s["cell_vertex_num"], s["cell_vertices"], t.Lx, t.Ly)
        assert np.allclose(ap, ref, rtol=1e-11, atol=1e-12)
        cand, win = sim.debug_t1()
        bc, bw = brute_force_t1(s, t.Lx, t.Ly, p["l_c"], t.S)
        assert [tuple(x) for x in cand.tolist()] == bc
        assert [tuple(x) for x in win.tolist()] == bw
        F, _ = sim.compute_forces()
        assert np.abs(F.sum(axis=0)).max() < 1e-10
        assert np.isfinite(s["pos"]).all()
    st = sim.get_state()["stats"]
    total_flips = st["t1_flips"]
    assert total_flips > 0, "the step-0 burst must produce flips"
    assert st["t1_candidates"] == st["t1_flips"] + st["t1_blocked"]
    assert st["error"] == 0


def test_many_flips_keep_invariants_larger_system():
    """configs[1] through the step-0 burst (hundreds of flips, conflicts included)."""
    t = w.config_tiling(1)
    p = w.config_params(1)
    sim = oracle.from_tiling(t, **p)
    s0 = sim.get_state()
    bc, bw = brute_force_t1(s0, t.Lx, t.Ly, p["l_c"], t.S)
    cand, win = sim.debug_t1()
    assert [tuple(x) for x in cand.tolist()] == bc and [tuple(x) for x in win.tolist()] == bw
    assert len(bw) < len(bc), "the Voronoi start must exercise the conflict rule"
    # no two winners share a cell
    used = set()
    for v, wv in bw:
        cells = set(edge_cells_from_rows(s0["cell_vertex_num"], s0["cell_vertices"], s0["vertex_cell_neighbors"], v, wv))
        assert not (cells & used)
        used |= cells
    sim.step(20)
    s = sim.get_state()
    h.check_topology(s["cell_vertex_num"], s["cell_vertices"], s["vertex_neighbors"], s["vertex_cell_neighbors"])
    ap = sim.geometry()
    assert abs(ap[:, 0].sum() - t.Lx * t.Ly) <= 1e-12 * t.Lx * t.Ly
    assert s["stats"]["t1_flips"] > 100


# ---- NEXT-1: the paper's own rule, T1 passes repeated until no candidate remains ----

def test_repeated_passes_resolve_a_conflict_chain_within_one_step():
    """The chain e1 < e2 < e3 of test_conflict_chain...: one pass flips e1 only; with repeated
    passes the blocked candidates flip in later passes of the SAME step, unless an earlier flip
    has already lengthened them, and the step ends at a fixed point of the rule."""
    l_c = 0.04
    t = w.hex_tiling(8, 6, a=1.0)
    row = t.cell_vertices[20, :6]
    pos = t.pos.copy()
    edges = [(int(row[0]), int(row[1])), (int(row[2]), int(row[3])), (int(row[4]), int(row[5]))]
    tt = t.copy()
    for a, b in edges:
        tt.pos = pos
        pos, _, _ = shrink_edge(tt, min(a, b), max(a, b), 0.5 * l_c)
    # K_A = K_P = v0 = 0: the step moves nothing, it only runs the T1 stage
    kw = dict(l_c=l_c, KA=0.0, KP=0.0, v0=0.0, Dr=0.0, dt=0.01)
    one = oracle.from_tiling(t, **kw)
    one.set_positions(pos)
    one.step(1)
    many = oracle.from_tiling(t, t1_max_passes=8, **kw)
    many.set_positions(pos)
    many.step(1)
    s1, sm = one.get_state()["stats"], many.get_state()["stats"]
    assert s1["t1_flips"] == 1 and s1["t1_blocked"] == 2
    assert sm["t1_flips"] >= 2 and sm["t1_flips"] > s1["t1_flips"]
    cand, _ = many.debug_t1()
    assert len(cand) == 0, "repeat-until-none must end at a fixed point of the rule"
    cand1, _ = one.debug_t1()
    assert len(cand1) > 0, "the single pass leaves the blocked candidates short"
    s = many.get_state()
    h.check_topology(s["cell_vertex_num"], s["cell_vertices"], s["vertex_neighbors"], s["vertex_cell_neighbors"])


def test_repeated_passes_on_a_voronoi_start():
    """configs[0] and configs[1]: with enough passes no candidate survives any step, every
    invariant of the single-pass rule still holds, and the first pass of every step is the
    single-pass rule itself (same candidates, same winners from the same state)."""
    for k, steps in ((0, 30), (1, 8)):
        t = w.config_tiling(k)
        p = w.config_params(k)
        sim = oracle.from_tiling(t, t1_max_passes=50, **p)
        ref = oracle.from_tiling(t, **p)
        # step 0 from the identical state: the repeated rule flips at least the single-pass winners
        sim.step(1)
        ref.step(1)
        assert sim.get_state()["stats"]["t1_flips"] >= ref.get_state()["stats"]["t1_flips"] > 0
        for _ in range(steps):
            sim.step(1)
            s = sim.get_state()
            cand, _ = sim.debug_t1()
            assert len(cand) == 0
            h.check_topology(s["cell_vertex_num"], s["cell_vertices"], s["vertex_neighbors"], s["vertex_cell_neighbors"])
            ap = sim.geometry()
            assert abs(ap[:, 0].sum() - t.Lx * t.Ly) <= 1e-12 * t.Lx * t.Ly
        st = sim.get_state()["stats"]
        assert st["t1_candidates"] == st["t1_flips"] + st["t1_blocked"] and st["error"] == 0


def test_one_pass_is_the_default_and_equals_max_passes_one():
    t = w.config_tiling(0)
    p = w.config_params(0)
    a = oracle.from_tiling(t, **p)
    b = oracle.from_tiling(t, t1_max_passes=1, **p)
    a.step(40)
    b.step(40)
    sa, sb = a.get_state(), b.get_state()
    assert np.array_equal(sa["pos"], sb["pos"]) and np.array_equal(sa["cell_vertices"], sb["cell_vertices"])


def pointing_edges(state, E):
    """edges (u, w) that have cell E as an END cell: u runs over E's row, w is u's neighbour outside E
    (slot convention R12: with vc[u][k] == E the row neighbours are vn[u][k], vn[u][k+1])"""
    vn, vc = state["vertex_neighbors"], state["vertex_cell_neighbors"]
    out = []
    for u in state["cell_vertices"][E, :state["cell_vertex_num"][E]]:
        k = vc[u].tolist().index(E)
        out.append((int(u), int(vn[u][(k + 2) % 3])))
    return out


def overflow_on_a_later_pass_case(l_c=0.04):
    """Hexagons with S = 8.  Cell E first gains a vertex (7 = S - 1); then two edges that both have E
    as an end cell are short: they conflict through E, the smaller key flips in pass 1 (E reaches
    S), and the other one is short, otherwise eligible, and rejected for overflow in pass 2."""
    t = w.hex_tiling(6, 4, a=1.0, S=8)
    E = 9
    kw = dict(l_c=l_c, KA=0.0, KP=0.0, v0=0.0, Dr=0.0, dt=0.01)
    sim = oracle.from_tiling(t, **kw)
    e0 = pointing_edges(sim.get_state(), E)[2]
    pos, _, _ = shrink_edge(t, min(e0), max(e0), 0.5 * l_c)
    sim.set_positions(pos)
    sim.t1_pass()
    s = sim.get_state()
    assert s["cell_vertex_num"][E] == 7
    tt = w.Tiling(t.Lx, t.Ly, t.S, s["pos"], s["cell_vertex_num"], s["cell_vertices"], s["vertex_neighbors"],
                  s["vertex_cell_neighbors"], s["theta"])
    touched = set(e0) | set(s["vertex_neighbors"][list(e0)].ravel().tolist())   # the flipped edge and its star
    far = [e for e in pointing_edges(s, E) if e[0] not in touched and e[1] not in touched]
    assert len(far) >= 2
    ea, eb = far[0], far[-1]
    for a, b in (ea, eb):
        tt.pos, _, _ = shrink_edge(tt, min(a, b), max(a, b), 0.5 * l_c)
    return tt, kw, E, sorted([tuple(sorted(ea)), tuple(sorted(eb))])


def test_repeated_passes_count_the_first_pass_and_raise_overflow_on_any_pass():
    """Reading of DESIGN.md section 9: t1_short and overflow_rejects are statistics of the step's
    first pass; the sticky error bit 2 ("a flip was suppressed because a row would exceed S") is
    raised by whichever pass sees it first, also a repeated one."""
    tt, kw, E, (first, second) = overflow_on_a_later_pass_case()
    chk = oracle.from_tiling(tt, **kw)
    cand, win = chk.debug_t1()
    assert [tuple(x) for x in cand.tolist()] == [first, second] and [tuple(x) for x in win.tolist()] == [first]
    many = oracle.from_tiling(tt, t1_max_passes=4, **kw)
    many.step(1)
    s = many.get_state()
    st = s["stats"]
    assert s["cell_vertex_num"][E] == 8
    assert st["t1_short"] == 2 and st["t1_candidates"] == 2 and st["t1_flips"] == 1 and st["t1_blocked"] == 1
    assert st["overflow_rejects"] == 0          # first-pass statistic: pass 1 rejected nothing
    assert st["error"] == 2                      # pass 2 suppressed the second edge: E is full
    cand, _ = many.debug_t1()
    assert len(cand) == 0
    # one pass per step: the overflow is seen (and counted) by the first pass of the NEXT step
    one = oracle.from_tiling(tt, **kw)
    one.step(1)
    assert one.get_state()["stats"]["error"] == 0 and one.get_state()["stats"]["overflow_rejects"] == 0
    one.step(1)
    st = one.get_state()["stats"]
    assert st["error"] == 2 and st["overflow_rejects"] == 1 and st["t1_short"] == 3 and st["t1_flips"] == 1


def test_an_edge_whose_end_cells_coincide_does_not_flip():
    """R10, "the four cells are distinct" (a reading: the paper is silent).  In a valid tiling E1, E2 never equal L
    or R (a vertex has three distinct cells) and L != R for cells narrower than half the box, so the clause is
    about E1 == E2: one cell touching both ends of an edge it does not contain.  tests/horseshoe.py reaches such a
    tiling from the 4 x 4 hexagonal torus by T1s and this test first checks it with the independent list checker.
    The edge is the only short one and passes every other clause (L, R have more than three vertices, E has room):
    it is counted as short, is no candidate, and the pass changes nothing.  Fails when the clause is deleted."""
    from tests import horseshoe as hs
    t, (v1, v2, cL, cR, cE) = hs.build()
    h.check_topology(t.cell_vertex_num, t.cell_vertices, t.vertex_neighbors, t.vertex_cell_neighbors)
    assert len({cL, cR, cE}) == 3
    rows = [set(t.cell_vertices[c, :t.cell_vertex_num[c]].tolist()) for c in (cL, cR, cE)]
    assert {v1, v2} <= rows[0] and {v1, v2} <= rows[1] and {v1, v2} <= rows[2]      # E holds both ends ...
    row = t.cell_vertices[cE, :t.cell_vertex_num[cE]].tolist()
    i1, n = row.index(v1), len(row)
    assert row[(i1 + 1) % n] != v2 and row[(i1 - 1) % n] != v2                       # ... but not the edge
    d = h.min_image(t.pos[v2] - t.pos[v1], np.array([t.Lx, t.Ly]))
    assert np.hypot(*d) < hs.PARAMS["l_c"]
    o = oracle.from_tiling(t, **hs.PARAMS)
    before = o.get_state()
    cand, win = o.debug_t1()
    assert len(cand) == 0 and len(win) == 0
    o.t1_pass()
    after = o.get_state()
    for key in ("cell_vertex_num", "cell_vertices", "vertex_neighbors", "vertex_cell_neighbors", "pos"):
        assert np.array_equal(before[key], after[key]), key
    st = after["stats"]
    assert st["t1_short"] == 1 and st["t1_candidates"] == 0 and st["t1_flips"] == 0 and st["error"] == 0
