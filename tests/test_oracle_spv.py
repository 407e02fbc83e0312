"""Pins of the SPV oracle (oracle/spv.py): the GPU-only parts of one self-propelled-Voronoi step on a fixed
triangulation (App. A.2).  None of these compares the oracle with itself: the generator's
Voronoi vertices, equidistance, central finite differences, lattice symmetry, closed forms of Eq. 3 and a
brute-force global circumcircle test."""
import numpy as np
import pytest

import oracle
from oracle import spv
from paper_1702_02939_b200 import workloads as w
from tests import helpers as h


def hex_centres(t):
    """centres of the regular hexagons of hex_tiling: mean of the unwrapped corners"""
    L = np.array([t.Lx, t.Ly])
    out = np.zeros((t.N, 2))
    for c in range(t.N):
        p0 = t.pos[t.cell_vertices[c, 0]]
        d = t.pos[t.cell_vertices[c, :6]] - p0
        d -= L * np.rint(d / L)
        out[c] = np.mod(p0 + d.mean(axis=0), L)
    return out


def test_circumcentres_of_a_voronoi_start_are_the_generators_vertices():
    """the tiling generator (tiling.cpp, independent code) places every vertex at the circumcentre of its
    three generating points: the oracle's circumcentres of those points must reproduce them, and each
    must be equidistant from its three corners"""
    for N, L, seed in ((64, 8.0, 1), (1024, 32.0, 5)):
        t = w.voronoi_tiling(N, L, seed)
        o = spv.SpvOracle(t, t.points)
        hv, ap = o.geometry()
        d = hv - t.pos
        d -= L * np.rint(d / L)
        assert np.abs(d).max() < 1e-9
        dist = np.stack([np.linalg.norm(h.min_image(hv - t.points[t.vertex_cell_neighbors[:, k]], L), axis=1) for k in range(3)], axis=1)
        assert np.abs(dist - dist[:, :1]).max() < 1e-11
        assert abs(ap[:, 0].sum() - L * L) < 1e-9 * L * L
        # areas and perimeters are those of the AVM oracle on the generator's own vertices
        ap_ref = oracle.from_tiling(t, **w.config_params(0)).geometry()
        assert np.abs(ap - ap_ref).max() < 1e-8


def test_circumcentre_jacobian_against_central_differences():
    t = w.voronoi_tiling(64, 8.0, 3)
    o = spv.SpvOracle(t, t.points)
    J = o.dh_dr()
    eps = 1e-6
    rng = np.random.default_rng(0)
    for v in rng.choice(t.V, 12, replace=False):
        for k in range(3):
            c = t.vertex_cell_neighbors[v, k]
            for a in range(2):
                rp, rm = t.points.copy(), t.points.copy()
                rp[c, a] += eps
                rm[c, a] -= eps
                dh = h.min_image(o.circumcentres(rp)[v] - o.circumcentres(rm)[v], 8.0) / (2 * eps)
                assert np.abs(dh - J[v, k, :, a]).max() < 1e-6 * max(1.0, np.abs(J[v, k]).max())


@pytest.mark.parametrize("params", [dict(KA=1.0, KP=1.0, A0=1.0, P0=3.8), dict(KA=1.0, KP=0.0, A0=0.7, P0=3.0), dict(KA=0.0, KP=1.0, A0=1.0, P0=4.2)])
def test_forces_against_central_differences_of_the_energy(params):
    """F_i = -dE/dr_i (Eq. 2 with the sign of Eq. A6), E = Eq. 1 on the Voronoi tiling of the cells"""
    t = w.voronoi_tiling(48, 7.0, 11)
    o = spv.SpvOracle(t, t.points, **params)
    F = o.forces()
    eps = 1e-5
    rms = np.sqrt((F ** 2).sum(1).mean())
    for c in range(0, t.N, 3):
        for a in range(2):
            rp, rm = t.points.copy(), t.points.copy()
            rp[c, a] += eps
            rm[c, a] -= eps
            fd = -(o.energy(rp) - o.energy(rm)) / (2 * eps)
            assert abs(fd - F[c, a]) < 1e-6 * max(abs(F[c, a]), rms), (c, a, fd, F[c, a])


def test_force_sets_sum_to_the_force_and_net_force_vanishes():
    t = w.voronoi_tiling(256, 16.0, 2)
    o = spv.SpvOracle(t, t.points, KA=1.0, KP=1.0, A0=1.0, P0=3.8)
    f = o.force_sets()
    F = o.forces()
    assert f.shape == (t.N, t.S, 2)
    assert np.abs(f.sum(axis=1) - F).max() < 1e-12
    used = np.arange(t.S)[None, :] < t.cell_vertex_num[:, None]
    assert np.abs(f[~used]).max() == 0.0
    assert np.abs(F.sum(axis=0)).max() < 1e-9          # translation invariance of E
    assert np.abs(F).max() > 0.1


def test_triangular_lattice_feels_no_force():
    t = w.hex_tiling(6, 6, a=0.7)
    r = hex_centres(t)
    for P0 in (3.0, 3.8):
        o = spv.SpvOracle(t, r, KA=1.0, KP=1.0, A0=1.0, P0=P0)
        hv, ap = o.geometry()
        assert np.abs(ap[:, 0] - 1.5 * np.sqrt(3.0) * 0.49).max() < 1e-12
        assert np.abs(o.forces()).max() < 1e-10


def test_eq3_pure_self_propulsion_and_director_noise():
    """K_A = K_P = 0: every cell moves by dt v0 (cos theta, sin theta) with the director of the start of the
    step (Eq. 3); the directors then take the Philox-keyed noise of PAPER.md:50"""
    t = w.voronoi_tiling(64, 8.0, 1)
    p = dict(KA=0.0, KP=0.0, v0=0.3, Dr=1.5, dt=0.01, seed=9)
    o = spv.SpvOracle(t, t.points, **p)
    th0 = o.theta.copy()
    o.step(1)
    d = h.min_image(o.r - t.points, 8.0)
    assert np.abs(d - 0.01 * 0.3 * np.stack([np.cos(th0), np.sin(th0)], axis=1)).max() < 1e-14
    th1 = th0 + np.sqrt(2 * 1.5 * 0.01) * oracle.director_noise(9, 0, 0, t.N)
    assert np.array_equal(o.theta, th1)
    o.step(1)
    d2 = h.min_image(o.r - t.points, 8.0) - d
    assert np.abs(d2 - 0.01 * 0.3 * np.stack([np.cos(th1), np.sin(th1)], axis=1)).max() < 1e-14


def test_eq3_mobility_scales_the_force_term():
    """Eq. 3: dr_i/dt = mu F_i + v0 n_i.  A passive step (v0 = 0) with mu = 0.37 displaces every cell
    by dt mu F(r0) (F from the force routine that central differences of E pin above), and, independently of that
    routine, the energy drops at the rate mu |F|^2: (E0 - E1) / (dt sum |F|^2) -> mu for a small step, with |F|^2
    taken from central differences of E.  Fails when the step drops mu or applies it to the propulsion term."""
    mu, dt = 0.37, 1e-7
    t = w.voronoi_tiling(64, 8.0, 4)
    o = spv.SpvOracle(t, t.points, KA=1.0, KP=1.0, A0=1.0, P0=3.6, v0=0.0, mu=mu, dt=dt)
    r0, F0, e0 = o.r.copy(), o.forces(), o.energy()
    o.step(1)
    d = h.min_image(o.r - r0, 8.0)
    assert np.abs(d - dt * mu * F0).max() < 1e-14
    # |F|^2 from central differences of the energy, not from forces()
    eps, g2 = 1e-6, 0.0
    for i in range(t.N):
        for a in range(2):
            rp, rm = r0.copy(), r0.copy()
            rp[i, a] += eps
            rm[i, a] -= eps
            g2 += ((o.energy(rp) - o.energy(rm)) / (2 * eps)) ** 2
    assert abs((e0 - o.energy()) / (dt * g2) - mu) < 2e-3 * mu
    # the propulsion term does not carry mu: active step, no forces
    a = spv.SpvOracle(t, t.points, KA=0.0, KP=0.0, v0=0.3, Dr=0.0, mu=mu, dt=0.01)
    th = a.theta.copy()
    a.step(1)
    assert np.abs(h.min_image(a.r - t.points, 8.0) - 0.01 * 0.3 * np.stack([np.cos(th), np.sin(th)], axis=1)).max() < 1e-14


def test_passive_spv_descends_the_energy():
    t = w.voronoi_tiling(64, 8.0, 4)
    o = spv.SpvOracle(t, t.points, KA=1.0, KP=1.0, A0=1.0, P0=3.6, v0=0.0, dt=2e-5)   # a Poisson-Voronoi start is stiff (max |F| ~ 90): small dt
    e = [o.energy()]
    for _ in range(10):
        o.step(1)
        e.append(o.energy())
    assert all(b < a for a, b in zip(e, e[1:]))


def test_local_circumcircle_verdict_equals_the_brute_force_one():
    """a Voronoi start is Delaunay: nothing fails.  After random displacements of growing size the local test
    (the cell opposite each edge) says "needs repair" exactly when the brute-force test over ALL cells does,
    and every triangle it flags is flagged by brute force too (local-Delaunay lemma, reading S2)."""
    t = w.voronoi_tiling(100, 10.0, 6)
    o = spv.SpvOracle(t, t.points)
    failed, margin, opp = o.test_triangulation()
    assert not failed.any() and not o.test_triangulation_global().any()
    assert margin.min() > 0
    rng = np.random.default_rng(1)
    seen_bad = 0
    for amp in (1e-6, 1e-5, 1e-4, 1e-3, 3e-3, 0.01, 0.03, 0.1, 0.3):
        for rep in range(3):
            r = np.mod(t.points + amp * rng.standard_normal(t.points.shape), 10.0)
            failed, margin, opp = o.test_triangulation(r)
            bad = o.test_triangulation_global(r)
            assert failed.any() == bad.any()
            assert not (failed.any(axis=1) & ~bad).any()
            seen_bad += int(bad.any())
    assert 3 < seen_bad < 24          # both verdicts occur (27 perturbations)
