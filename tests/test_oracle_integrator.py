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
