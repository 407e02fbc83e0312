"""Pins for the oracle's integrator (PAPER.md:56 Eq. 4, :50 director noise, :104 order).
Closed forms and statistical laws only; SURVEY.md §8(c) "Integrator" pin row."""
import numpy as np

import oracle
from paper_1702_02939_b200 import workloads as w
from tests import helpers as h


def test_pure_activity_translates_every_vertex():
    """K_A = K_P = 0, D_r = 0, uniform theta: every vertex moves by v0*dt*(cos, sin) per step
    (Eq. 4 with n = 3 identical directors), wrapping through the box."""
    th0 = 0.7
    t = w.hex_tiling(6, 4, a=1.0, theta=np.full(24, th0))
    v0, dt, n = 0.3, 0.01, 250
    sim = oracle.from_tiling(t, KA=0.0, KP=0.0, v0=v0, Dr=0.0, dt=dt, l_c=0.0, seed=1)
    sim.step(n)
    s = sim.get_state()
    expect = t.pos + n * v0 * dt * np.array([np.cos(th0), np.sin(th0)])
    d = s["pos"] - expect
    d[:, 0] = h.min_image(d[:, 0], t.Lx); d[:, 1] = h.min_image(d[:, 1], t.Ly)
    assert np.abs(d).max() < 1e-12
    assert (s["pos"] >= 0).all() and (s["pos"][:, 0] < t.Lx).all() and (s["pos"][:, 1] < t.Ly).all()
    assert np.array_equal(s["theta"], np.full(24, th0))
    assert s["stats"]["step"] == n


def test_mean_director_is_average_of_three_cells():
    """Eq. 4: activity on a vertex is (v0/3) * sum of its three cells' unit directors."""
    t = w.config_tiling(0)
    v0, dt = 0.2, 0.01
    sim = oracle.from_tiling(t, KA=0.0, KP=0.0, v0=v0, Dr=0.0, dt=dt, l_c=0.0)
    sim.step(1)
    s = sim.get_state()
    n = np.stack([np.cos(t.theta), np.sin(t.theta)], axis=1)
    drift = v0 / 3.0 * n[t.vertex_cell_neighbors].sum(axis=1) * dt
    d = s["pos"] - (t.pos + drift)
    d[:, 0] = h.min_image(d[:, 0], t.Lx); d[:, 1] = h.min_image(d[:, 1], t.Ly)
    assert np.abs(d).max() < 1e-14


def test_passive_dynamics_is_gradient_descent():
    """v0 = 0, D_r = 0, no T1: E decreases monotonically for small dt, and the first step moves
    each vertex by mu*dt*F (overdamped Euler)."""
    t = w.config_tiling(0)
    p = dict(w.config_params(0), v0=0.0, Dr=0.0, l_c=0.0, dt=1e-3, mu=0.5)
    sim = oracle.from_tiling(t, **p)
    F, _ = sim.compute_forces()
    E = [sim.energy()]
    sim.step(1)
    s = sim.get_state()
    d = s["pos"] - (t.pos + p["mu"] * p["dt"] * F)
    d[:, 0] = h.min_image(d[:, 0], t.Lx); d[:, 1] = h.min_image(d[:, 1], t.Ly)
    assert np.abs(d).max() < 1e-14
    for _ in range(50):
        E.append(sim.energy())
        sim.step(1)
    assert all(b < a for a, b in zip(E, E[1:]))


def test_director_diffusion_variance():
    """Var(theta(t) - theta(0)) = 2 D_r t (Euler-Maruyama of d theta = eta, <eta eta> = 2 D_r)."""
    t = w.config_tiling(1)
    Dr, dt, n = 0.8, 0.01, 40
    sim = oracle.from_tiling(t, KA=0.0, KP=0.0, v0=0.0, Dr=Dr, dt=dt, l_c=0.0, seed=7)
    sim.step(n)
    dth = sim.get_state()["theta"] - t.theta
    var = dth.var()
    expect = 2 * Dr * dt * n
    assert abs(var / expect - 1.0) < 4.0 * np.sqrt(2.0 / t.N)
    assert abs(dth.mean()) < 4.0 * np.sqrt(expect / t.N)


def test_director_update_uses_step_and_cell_keys():
    """theta_c(s+1) - theta_c(s) = sqrt(2 Dr dt) * xi(seed, s, c) with the step counter starting
    at step0 (resume must be bit-identical, SURVEY §5 checkpoint row)."""
    t = w.config_tiling(0)
    Dr, dt, seed = 1.0, 0.01, 7
    sim = oracle.from_tiling(t, KA=0.0, KP=0.0, v0=0.0, Dr=Dr, dt=dt, l_c=0.0, seed=seed, step0=41)
    sim.step(2)
    th = sim.get_state()["theta"]
    amp = np.sqrt(2 * Dr * dt)
    expect = t.theta + amp * oracle.director_noise(seed, 41, 0, t.N)
    expect = expect + amp * oracle.director_noise(seed, 42, 0, t.N)
    assert np.array_equal(th, expect)


def test_resume_is_bit_identical():
    t = w.config_tiling(0)
    p = w.config_params(0)
    a = oracle.from_tiling(t, **p)
    a.step(60)
    b = oracle.from_tiling(t, **p)
    b.step(25)
    s = b.get_state()
    c = oracle.OracleSim(s["pos"], s["cell_vertex_num"], s["cell_vertices"], s["vertex_neighbors"],
                         s["vertex_cell_neighbors"], s["theta"], **dict(p, step0=25))
    c.step(35)
    sa, sc = a.get_state(), c.get_state()
    for k in ("pos", "theta", "cell_vertices", "vertex_neighbors", "vertex_cell_neighbors", "cell_vertex_num"):
        assert np.array_equal(sa[k], sc[k]), k


def test_vertices_move_with_start_of_step_directors():
    """R7 (PAPER.md:104 "first move the vertices and then update the cell directors"; Eq. 4, :56):
    with K_A = K_P = 0, v0 > 0 and Dr > 0 the displacement of a step is dt*v0/3 * sum n(theta) with
    theta taken at the START of that step, and the next step uses the rotated directors
    theta1 = theta0 + sqrt(2 Dr dt) xi(seed, 0, c).  A swapped move/rotate order fails both halves."""
    t = w.config_tiling(0)
    v0, dt, Dr, seed = 0.7, 0.01, 2.0, 11
    sim = oracle.from_tiling(t, KA=0.0, KP=0.0, v0=v0, Dr=Dr, dt=dt, l_c=0.0, seed=seed)
    th0 = t.theta
    th1 = th0 + np.sqrt(2 * Dr * dt) * oracle.director_noise(seed, 0, 0, t.N)
    vc = t.vertex_cell_neighbors

    def drift(th):
        n = np.stack([np.cos(th), np.sin(th)], axis=1)
        return dt * v0 / 3.0 * n[vc].sum(axis=1)

    def mi_diff(a, b):
        d = a - b
        return np.stack([h.min_image(d[:, 0], t.Lx), h.min_image(d[:, 1], t.Ly)], axis=1)

    sim.step(1)
    s1 = sim.get_state()
    assert np.abs(mi_diff(s1["pos"], t.pos) - drift(th0)).max() < 1e-14
    assert np.abs(drift(th1) - drift(th0)).max() > 1e-4           # the two readings are far apart
    assert np.abs(mi_diff(s1["pos"], t.pos) - drift(th1)).max() > 1e-4
    assert np.array_equal(s1["theta"], th1)
    sim.step(1)
    s2 = sim.get_state()
    assert np.abs(mi_diff(s2["pos"], s1["pos"]) - drift(th1)).max() < 1e-14
    th2 = th1 + np.sqrt(2 * Dr * dt) * oracle.director_noise(seed, 1, 0, t.N)
    assert np.abs(mi_diff(s2["pos"], s1["pos"]) - drift(th2)).max() > 1e-4


def test_topology_is_tested_on_the_moved_positions():
    """R6 ("with the forces in hand the degrees of freedom can be displaced ...
    the next challenge is determining whether the cellular topology needs to be updated"; :104-108):
    an edge that is longer than l_c at the start of the step and is brought below l_c by that
    step's move flips in that very step; with the T1 pass before the move it would not."""
    from tests.test_oracle_t1 import edge_cells_from_rows, shrink_edge
    l_c, dt, v0 = 0.04, 0.01, 0.9
    t = w.hex_tiling(6, 4, a=1.0)
    v1 = 7
    v2 = int(t.vertex_neighbors[v1, 1])
    lo, hi = min(v1, v2), max(v1, v2)
    L, R, E1, E2 = edge_cells_from_rows(t.cell_vertex_num, t.cell_vertices, t.vertex_cell_neighbors, lo, hi)
    closing = dt * 2.0 * v0 / 3.0            # the end cells' directors point at each other along the edge
    start_len = l_c + 0.5 * closing
    pos, m, u = shrink_edge(t, lo, hi, start_len)
    theta = np.zeros(t.N)
    theta[E1] = np.arctan2(u[1], u[0])        # E1 holds lo: push lo towards hi
    theta[E2] = np.arctan2(-u[1], -u[0])      # E2 holds hi: push hi towards lo
    theta[L] = theta[R] = 0.3                 # shared by both endpoints: no relative motion
    tt = w.Tiling(t.Lx, t.Ly, t.S, pos, t.cell_vertex_num, t.cell_vertices, t.vertex_neighbors,
                  t.vertex_cell_neighbors, theta)
    sim = oracle.from_tiling(tt, KA=0.0, KP=0.0, v0=v0, Dr=0.0, dt=dt, l_c=l_c)
    cand, _ = sim.debug_t1()
    assert len(cand) == 0                     # nothing is short before the move
    sim.step(1)
    s = sim.get_state()
    assert s["stats"]["t1_short"] == 1 and s["stats"]["t1_flips"] == 1
    assert h.cells_adjacent(s["cell_vertices"], s["cell_vertex_num"], E1, E2)
    d = s["pos"][hi] - s["pos"][lo]
    assert abs(np.hypot(h.min_image(d[0], t.Lx), h.min_image(d[1], t.Ly)) - 1.5 * l_c) < 1e-14
    # the length the pass saw was start_len - closing < l_c: one more identical system, T1 off
    ref = oracle.from_tiling(tt, KA=0.0, KP=0.0, v0=v0, Dr=0.0, dt=dt, l_c=0.0)
    ref.step(1)
    r = ref.get_state()["pos"]
    d = r[hi] - r[lo]
    assert abs(np.hypot(h.min_image(d[0], t.Lx), h.min_image(d[1], t.Ly)) - (start_len - closing)) < 1e-13


# ---- NEXT-2: mean-square displacement of the vertices (unwrapped positions) ----

def test_msd_of_pure_activity_is_the_closed_form_through_the_box():
    """K_A = K_P = 0, D_r = 0, uniform theta: every vertex has moved by n*v0*dt along the director, so
    the mean-square displacement is (n v0 dt)^2 exactly, however often the box wrapped; a reset
    restarts it from zero."""
    th0 = 2.1
    t = w.hex_tiling(6, 4, a=1.0, theta=np.full(24, th0))
    v0, dt, n = 0.8, 0.01, 1500                      # 12 length units: more than one box length (10.4 x 6)
    sim = oracle.from_tiling(t, KA=0.0, KP=0.0, v0=v0, Dr=0.0, dt=dt, l_c=0.0)
    assert sim.msd() == 0.0
    sim.step(n)
    assert abs(sim.msd() - (n * v0 * dt) ** 2) < 1e-9 * (n * v0 * dt) ** 2
    sim.msd_reset()
    assert sim.msd() == 0.0
    sim.step(10)
    assert abs(sim.msd() - (10 * v0 * dt) ** 2) < 1e-12


def test_msd_counts_the_repositioning_of_a_t1():
    """one hand-built flip and nothing else moving: the two end points go from +-len/2 along the edge to
    +-0.75 l_c across it (R9), so MSD = 2 ((len/2)^2 + (0.75 l_c)^2) / V"""
    from tests.test_oracle_t1 import shrink_edge
    l_c = 0.04
    t = w.hex_tiling(6, 4, a=1.0)
    v1, v2 = 7, int(t.vertex_neighbors[7, 1])
    ln = 0.5 * l_c
    pos, _, _ = shrink_edge(t, min(v1, v2), max(v1, v2), ln)
    sim = oracle.from_tiling(t, KA=0.0, KP=0.0, v0=0.0, Dr=0.0, dt=0.01, l_c=l_c)
    sim.set_positions(pos)
    sim.step(1)
    assert sim.get_state()["stats"]["t1_flips"] == 1
    assert abs(sim.msd() - 2 * ((0.5 * ln) ** 2 + (0.75 * l_c) ** 2) / t.V) < 1e-15


def test_msd_equals_an_independent_unwrapping_of_the_trajectory():
    """configs[0] with a large drift so that vertices cross the box: the oracle's MSD against numpy's
    accumulation of minimum-image differences between consecutive snapshots (valid because one step
    moves a vertex by far less than L/2)"""
    t = w.config_tiling(0)
    p = dict(w.config_params(0), v0=3.0, Dr=0.2)
    sim = oracle.from_tiling(t, **p)
    prev = t.pos.copy()
    U = np.zeros_like(prev)
    for _ in range(300):
        sim.step(1)
        cur = sim.get_state()["pos"]
        d = cur - prev
        U[:, 0] += h.min_image(d[:, 0], t.Lx)
        U[:, 1] += h.min_image(d[:, 1], t.Ly)
        prev = cur
    ref = (U ** 2).sum(axis=1).mean()
    assert np.abs((prev - t.pos) - U).max() > 0.5 * t.Lx        # some vertices really left through the box boundary
    assert abs(sim.msd() - ref) < 1e-10 * ref
    assert sim.get_state()["stats"]["t1_flips"] > 0
    assert abs(sim.observables()["msd"] - sim.msd()) == 0.0


def test_the_two_halves_of_a_step_are_the_step():
    """oracle.step is step_move_and_rotate followed by step_topology_and_advance (the split only exposes
    the moved tiling before the topology update, PAPER.md:62-64 order): identical bits, and between the
    halves the step counter has not advanced, positions have moved and no flip has been counted."""
    t = w.config_tiling(0)
    p = w.config_params(0)
    a = oracle.from_tiling(t, **p)
    b = oracle.from_tiling(t, **p)
    for _ in range(30):
        a.step(1)
        before = b.get_state()
        b.step_move_and_rotate()
        mid = b.get_state()
        assert mid["stats"]["step"] == before["stats"]["step"]
        assert mid["stats"]["t1_flips"] == before["stats"]["t1_flips"]
        assert np.array_equal(mid["cell_vertices"], before["cell_vertices"])
        assert not np.array_equal(mid["pos"], before["pos"])
        b.step_topology_and_advance()
        sa, sb = a.get_state(), b.get_state()
        for key in ("pos", "theta", "cell_vertices", "cell_vertex_num", "vertex_neighbors", "vertex_cell_neighbors"):
            assert np.array_equal(sa[key], sb[key]), key
        assert sa["stats"] == sb["stats"]
    assert a.get_state()["stats"]["t1_flips"] > 0
