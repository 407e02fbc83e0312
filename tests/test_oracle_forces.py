"""Pins for the oracle's geometry, energy and forces (PAPER.md:39 Eq. 1, :154-169 Eq. A1-A5).

Nothing here compares the oracle with itself: closed forms for regular hexagons, central finite
differences of Eq. A1 (the energy is a different code path from the force), conservation laws,
and an independent numpy shoelace / scipy cross-check."""
import math

import numpy as np
import pytest

import oracle
from paper_1702_02939_b200 import workloads as w
from tests import helpers as h

PARAMS = dict(KA=1.0, KP=1.0, A0=1.0, P0=3.8)


def test_hexagon_closed_forms_and_zero_force():
    """Regular hexagons of side a: A = (3 sqrt3 / 2) a^2, P = 6a, and F = 0 on every vertex for
    any (A0, P0): three identical cells meet at 120 degrees (SURVEY 8(c) pins)."""
    for a, A0, P0 in [(1.0, 1.0, 3.8), (0.62, 1.0, 3.6), (0.9, 2.5, 1.0)]:
        t = w.hex_tiling(6, 4, a=a)
        sim = oracle.from_tiling(t, KA=1.3, KP=0.7, A0=A0, P0=P0)
        F, ap = sim.compute_forces()
        assert np.allclose(ap[:, 0], 1.5 * np.sqrt(3.0) * a * a, rtol=1e-13, atol=0)
        assert np.allclose(ap[:, 1], 6.0 * a, rtol=1e-13, atol=0)
        assert np.abs(F).max() <= 1e-12
        E = sim.energy()
        E_closed = t.N * (1.3 * (1.5 * np.sqrt(3.0) * a * a - A0) ** 2 + 0.7 * (6 * a - P0) ** 2)
        assert abs(E - E_closed) <= 1e-12 * max(1.0, E_closed)


def test_single_moved_vertex_in_hexagons_closed_form():
    """Move one vertex of a hexagonal tiling outward along an edge direction: the perimeter and
    area changes of the three cells have elementary closed forms (catches a wrong prev/next)."""
    a = 1.0
    t = w.hex_tiling(6, 4, a=a)
    v = 5
    nb = t.vertex_neighbors[v]
    d = t.pos[nb[0]] - t.pos[v]
    d[0] = h.min_image(d[0], t.Lx); d[1] = h.min_image(d[1], t.Ly)
    eps = 0.1
    pos = t.pos.copy()
    pos[v] += eps * d / np.linalg.norm(d)        # slide along edge to neighbour 0
    sim = oracle.from_tiling(t)
    sim.set_positions(np.mod(pos, [t.Lx, t.Ly]))
    ap = sim.geometry()
    A_hex = 1.5 * np.sqrt(3.0)
    cells = t.vertex_cell_neighbors[v]
    # each of the two cells containing edge (v, n0) loses the triangle (v_old, v_new, its other
    # neighbour of v); the cell opposite the edge gains both triangles; total area is conserved
    assert abs(ap[:, 0].sum() - t.Lx * t.Ly) < 1e-12 * t.Lx * t.Ly
    tri = 0.5 * eps * a * np.sin(2 * np.pi / 3)  # sides eps and a enclosing 120 degrees
    dA = ap[cells, 0] - A_hex
    assert np.allclose(sorted(dA), [-tri, -tri, 2 * tri], atol=1e-13)
    # perimeters: edge (v,n0) shortens by eps; the other two edges become sqrt(a^2+eps^2+a*eps)
    l2 = np.sqrt(a * a + eps * eps + a * eps)
    dP = ap[cells, 1] - 6 * a
    expect = sorted([(-eps) + (l2 - a), (-eps) + (l2 - a), 2 * (l2 - a)])
    assert np.allclose(sorted(dP), expect, atol=1e-13)


@pytest.mark.parametrize("N,L,seed", [(64, 8.0, 1), (100, 10.0, 3)])
def test_forces_match_finite_differences_of_energy(N, L, seed):
    """F = -dE/dh (Eq. A2) against central differences of Eq. A1, to 1e-6 relative."""
    t = w.voronoi_tiling(N, L, seed)
    sim = oracle.from_tiling(t, **PARAMS)
    F, ap0 = sim.compute_forces()
    rms = np.sqrt((F ** 2).sum(axis=1).mean())
    worst = 0.0
    others_checked = False
    for v in range(t.V):
        cells = t.vertex_cell_neighbors[v]
        # step well below the shortest incident edge (the perimeter has derivatives ~ 1/l^k) and a
        # 4th-order central stencil, so truncation stays far below the 1e-6 target
        dn = t.pos[t.vertex_neighbors[v]] - t.pos[v]
        lmin = np.hypot(h.min_image(dn[:, 0], t.Lx), h.min_image(dn[:, 1], t.Ly)).min()
        delta = min(1e-5, 1e-2 * lmin)
        g = np.zeros(2)
        for ax in range(2):
            e = {}
            for m in (-2, -1, 1, 2):
                pos = t.pos.copy()
                pos[v, ax] += m * delta
                pos[v, ax] %= (t.Lx, t.Ly)[ax]
                sim.set_positions(pos)
                ap = sim.geometry()
                # only the three cells of v change: difference their energies alone (less round-off)
                e[m] = np.sum(PARAMS["KA"] * (ap[cells, 0] - PARAMS["A0"]) ** 2 +
                              PARAMS["KP"] * (ap[cells, 1] - PARAMS["P0"]) ** 2)
                if not others_checked:
                    others = np.setdiff1d(np.arange(N), cells)
                    assert np.array_equal(ap[others], ap0[others])
                    others_checked = True
            g[ax] = (8 * (e[1] - e[-1]) - (e[2] - e[-2])) / (12 * delta)
        err = np.linalg.norm(F[v] + g) / max(np.linalg.norm(F[v]), rms)
        worst = max(worst, err)
    assert worst < 1e-6, worst


@pytest.mark.parametrize("k", [0, 1])
def test_conservation_laws_on_configs(k):
    t = w.config_tiling(k)
    p = w.config_params(k)
    sim = oracle.from_tiling(t, **p)
    F, ap = sim.compute_forces()
    L2 = t.Lx * t.Ly
    assert abs(ap[:, 0].sum() - L2) <= 1e-12 * L2                      # areas tile the box
    scale = np.abs(F).sum(axis=0)
    assert (np.abs(F.sum(axis=0)) <= 1e-10 * np.maximum(scale, 1.0)).all()   # translation invariance
    assert np.abs(F.sum(axis=0)).max() < 1e-10
    # geometry against an independent numpy shoelace
    ref = h.polygon_areas_numpy(t.pos, t.cell_vertex_num, t.cell_vertices, t.Lx, t.Ly)
    assert np.allclose(ap, ref, rtol=1e-12, atol=1e-13)


def test_forces_invariant_under_rigid_shift():
    """Shifting all positions by a vector (with wrap) must not change A, P or F: tests the
    minimum-image / wrap handling across the box boundary."""
    t = w.config_tiling(0)
    p = w.config_params(0)
    sim = oracle.from_tiling(t, **p)
    F0, ap0 = sim.compute_forces()
    rng = np.random.default_rng(0)
    for _ in range(5):
        shift = rng.uniform(0, t.Lx, size=2)
        sim.set_positions(np.mod(t.pos + shift, [t.Lx, t.Ly]))
        F, ap = sim.compute_forces()
        assert np.allclose(ap, ap0, rtol=1e-12, atol=1e-13)
        assert np.allclose(F, F0, rtol=0, atol=1e-11)


def test_force_of_area_and_perimeter_terms_separately():
    """K_P = 0: force is the pressure term only; for a single inflated cell pressure pushes its
    vertices outward.  K_A = 0 with P > P0: tension pulls neighbours together (sign pins)."""
    t = w.hex_tiling(6, 4, a=1.0)
    A_hex = 1.5 * np.sqrt(3.0)
    # all cells at preferred area except that A0 is smaller than A: every cell wants to shrink,
    # symmetric -> zero force; now enlarge one cell by moving one of its vertices outward
    c = 9
    v = t.cell_vertices[c, 0]
    polys = h.unwrapped_polygons(t.pos, t.cell_vertex_num, t.cell_vertices, t.Lx, t.Ly)
    centre = polys[c].mean(axis=0)
    out = polys[c][0] - centre
    out /= np.linalg.norm(out)
    pos = t.pos.copy()
    pos[v] = np.mod(pos[v] + 0.05 * out, [t.Lx, t.Ly])
    sim = oracle.from_tiling(t, KA=1.0, KP=0.0, A0=A_hex, P0=0.0)
    sim.set_positions(pos)
    F, ap = sim.compute_forces()
    assert ap[c, 0] > A_hex
    assert F[v] @ out < 0          # restoring: pushed back toward the centre of the enlarged cell
    sim2 = oracle.from_tiling(t, KA=0.0, KP=1.0, A0=0.0, P0=6.0)
    sim2.set_positions(pos)
    F2, ap2 = sim2.compute_forces()
    assert ap2[c, 1] > 6.0
    assert F2[v] @ out < 0         # line tension also restores


def test_energy_definition_has_no_half():
    """Eq. 1 has no 1/2: E for a single perturbed configuration recomputed from A, P in numpy."""
    t = w.config_tiling(0)
    p = w.config_params(0)
    sim = oracle.from_tiling(t, **p)
    ap = h.polygon_areas_numpy(t.pos, t.cell_vertex_num, t.cell_vertices, t.Lx, t.Ly)
    E = np.sum(p["KA"] * (ap[:, 0] - p["A0"]) ** 2 + p["KP"] * (ap[:, 1] - p["P0"]) ** 2)
    assert abs(sim.energy() - E) <= 1e-12 * E


def test_observables_closed_forms_on_hexagons_and_voronoi():
    """NEXT-2 pins: regular hexagons of side a have shape index 6a / sqrt(3 sqrt(3)/2 a^2) =
    3.72241943..., zero area variance and E = N [KA (A-A0)^2 + KP (P-P0)^2]; on a Voronoi tiling
    the areas sum to L^2, so the mean area is L^2 / N and the variance follows from the cells."""
    a = 0.8
    t = w.hex_tiling(6, 4, a=a)
    o = oracle.from_tiling(t, KA=1.3, KP=0.7, A0=1.0, P0=3.9)
    ob = o.observables()
    A, P = 1.5 * math.sqrt(3.0) * a * a, 6.0 * a
    assert abs(ob["mean_shape_index"] - 6.0 / math.sqrt(1.5 * math.sqrt(3.0))) < 1e-13
    assert abs(ob["mean_shape_index"] - 3.7224194364083982) < 1e-13
    assert abs(ob["area_variance"]) < 1e-13 and ob["n_nonpositive_area"] == 0
    assert abs(ob["area_min"] - A) < 1e-13 and abs(ob["area_max"] - A) < 1e-13
    assert abs(ob["energy"] - 24 * (1.3 * (A - 1.0) ** 2 + 0.7 * (P - 3.9) ** 2)) < 1e-11
    t = w.config_tiling(1)
    o = oracle.from_tiling(t, **w.config_params(1))
    ob = o.observables()
    L2 = t.Lx * t.Ly
    assert abs(ob["sum_area"] - L2) <= 1e-12 * L2
    ref = h.polygon_areas_numpy(t.pos, t.cell_vertex_num, t.cell_vertices, t.Lx, t.Ly)   # independent shoelace
    assert abs(ob["area_variance"] - ref[:, 0].var()) < 1e-12
    assert abs(ob["mean_shape_index"] - (ref[:, 1] / np.sqrt(ref[:, 0])).mean()) < 1e-12
    assert 0.2 < ob["area_variance"] < 0.35        # Poisson-Voronoi: var(A) / <A>^2 ~ 0.28


# ---- NEXT-4: per-cell preferred values A_{0,i}, P_{0,i} of Eq. 1 ----

def test_per_cell_targets_match_finite_differences_of_eq1():
    """heterogeneous A0_i, P0_i: F = -dE/dh against central differences of Eq. 1, whose energy
    is written out here with numpy from the oracle's geometry"""
    t = w.voronoi_tiling(64, 8.0, 5)
    rng = np.random.default_rng(0)
    A0 = rng.uniform(0.6, 1.4, t.N)
    P0 = rng.uniform(3.2, 4.2, t.N)
    sim = oracle.from_tiling(t, **PARAMS)
    sim.set_cell_targets(A0, P0)
    F, ap0 = sim.compute_forces()
    assert abs(sim.energy() - np.sum(PARAMS["KA"] * (ap0[:, 0] - A0) ** 2 + PARAMS["KP"] * (ap0[:, 1] - P0) ** 2)) < 1e-10
    rms = np.sqrt((F ** 2).sum(axis=1).mean())
    worst = 0.0
    for v in range(0, t.V, 3):
        cells = t.vertex_cell_neighbors[v]
        dn = t.pos[t.vertex_neighbors[v]] - t.pos[v]
        lmin = np.hypot(h.min_image(dn[:, 0], t.Lx), h.min_image(dn[:, 1], t.Ly)).min()
        delta = min(1e-5, 1e-2 * lmin)
        g = np.zeros(2)
        for ax in range(2):
            e = {}
            for m in (-2, -1, 1, 2):
                pos = t.pos.copy()
                pos[v, ax] += m * delta
                pos[v, ax] %= (t.Lx, t.Ly)[ax]
                sim.set_positions(pos)
                ap = sim.geometry()
                e[m] = np.sum(PARAMS["KA"] * (ap[cells, 0] - A0[cells]) ** 2 + PARAMS["KP"] * (ap[cells, 1] - P0[cells]) ** 2)
            g[ax] = (8 * (e[1] - e[-1]) - (e[2] - e[-2])) / (12 * delta)
        worst = max(worst, np.linalg.norm(F[v] + g) / max(np.linalg.norm(F[v]), rms))
    assert worst < 1e-6, worst
    # translation invariance survives heterogeneity
    sim.set_positions(t.pos)
    assert np.abs(sim.compute_forces()[0].sum(axis=0)).max() < 1e-10


def test_per_cell_targets_special_cases():
    """(i) arrays filled with the uniform values reproduce the uniform path bit for bit; (ii) with
    each cell's targets set to its own area and perimeter every force vanishes and E = 0;
    (iii) NULL, NULL restores the uniform values."""
    t = w.config_tiling(0)
    p = w.config_params(0)
    a = oracle.from_tiling(t, **p)
    b = oracle.from_tiling(t, **p)
    b.set_cell_targets(np.full(t.N, p["A0"]), np.full(t.N, p["P0"]))
    a.step(30)
    b.step(30)
    assert np.array_equal(a.get_state()["pos"], b.get_state()["pos"])
    c = oracle.from_tiling(t, **p)
    ap = c.geometry()
    c.set_cell_targets(ap[:, 0], ap[:, 1])
    assert np.abs(c.compute_forces()[0]).max() == 0.0 and c.energy() == 0.0
    c.set_cell_targets(None, None)
    assert np.array_equal(c.compute_forces()[0], oracle.from_tiling(t, **p).compute_forces()[0])


def test_per_cell_moduli_match_finite_differences_of_eq1():
    """heterogeneous K_{A,i}, K_{P,i} together with heterogeneous targets (Eq. 1, read with the
    moduli inside the sum): F = -dE/dh against central differences of the energy written out
    here with numpy from the oracle's geometry; uniform arrays reproduce the scalar path bit for bit;
    zero moduli on a cell switch that cell's contribution off."""
    t = w.voronoi_tiling(64, 8.0, 6)
    rng = np.random.default_rng(1)
    A0, P0 = rng.uniform(0.6, 1.4, t.N), rng.uniform(3.2, 4.2, t.N)
    KA, KP = rng.uniform(0.2, 3.0, t.N), rng.uniform(0.1, 2.0, t.N)
    sim = oracle.from_tiling(t, **PARAMS)
    sim.set_cell_targets(A0, P0)
    sim.set_cell_moduli(KA, KP)
    F, ap0 = sim.compute_forces()
    assert abs(sim.energy() - np.sum(KA * (ap0[:, 0] - A0) ** 2 + KP * (ap0[:, 1] - P0) ** 2)) < 1e-10
    rms = np.sqrt((F ** 2).sum(axis=1).mean())
    worst = 0.0
    for v in range(0, t.V, 3):
        cells = t.vertex_cell_neighbors[v]
        dn = t.pos[t.vertex_neighbors[v]] - t.pos[v]
        lmin = np.hypot(h.min_image(dn[:, 0], t.Lx), h.min_image(dn[:, 1], t.Ly)).min()
        delta = min(1e-5, 1e-2 * lmin)
        g = np.zeros(2)
        for ax in range(2):
            e = {}
            for m in (-2, -1, 1, 2):
                pos = t.pos.copy()
                pos[v, ax] += m * delta
                pos[v, ax] %= (t.Lx, t.Ly)[ax]
                sim.set_positions(pos)
                ap = sim.geometry()
                e[m] = np.sum(KA[cells] * (ap[cells, 0] - A0[cells]) ** 2 + KP[cells] * (ap[cells, 1] - P0[cells]) ** 2)
            g[ax] = (8 * (e[1] - e[-1]) - (e[2] - e[-2])) / (12 * delta)
        worst = max(worst, np.linalg.norm(F[v] + g) / max(np.linalg.norm(F[v]), rms))
    assert worst < 1e-6, worst
    sim.set_positions(t.pos)
    assert np.abs(sim.compute_forces()[0].sum(axis=0)).max() < 1e-10
    # uniform arrays = the scalar path, bit for bit, through T1s
    t0 = w.config_tiling(0)
    p = w.config_params(0)
    a, b = oracle.from_tiling(t0, **p), oracle.from_tiling(t0, **p)
    b.set_cell_moduli(np.full(t0.N, p["KA"]), np.full(t0.N, p["KP"]))
    a.step(30)
    b.step(30)
    assert np.array_equal(a.get_state()["pos"], b.get_state()["pos"])
    # a cell with zero moduli exerts no force: the force on a vertex then comes from its other cells only
    c = oracle.from_tiling(t0, **p)
    KA0, KP0 = np.full(t0.N, p["KA"]), np.full(t0.N, p["KP"])
    dead = int(t0.vertex_cell_neighbors[5, 0])
    KA0[dead] = KP0[dead] = 0.0
    c.set_cell_moduli(KA0, KP0)
    F1 = c.compute_forces()[0]
    far = np.array([v for v in range(t0.V) if dead not in t0.vertex_cell_neighbors[v]])
    assert np.array_equal(F1[far], a.__class__(t0.pos, t0.cell_vertex_num, t0.cell_vertices, t0.vertex_neighbors,
                                               t0.vertex_cell_neighbors, t0.theta, **p).compute_forces()[0][far])
    c.set_cell_moduli(None, None)
    assert np.array_equal(c.compute_forces()[0], oracle.from_tiling(t0, **p).compute_forces()[0])
