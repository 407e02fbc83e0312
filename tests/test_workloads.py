"""Pins for the seeded input generator (paper_1702_02939_b200/workloads): the periodic Voronoi
tiling is checked against scipy.spatial (library routine), brute force and Euler's formula.
DESIGN.md §"Input recipe"; SURVEY.md §8(c) R20 and the "Tiling generator" pin row."""
import numpy as np
import pytest

from paper_1702_02939_b200 import workloads as w
from tests import helpers as h


@pytest.mark.parametrize("N,L,seed", [(64, 8.0, 1), (300, 17.3, 11), (4096, 64.0, 2)])
def test_voronoi_invariants(N, L, seed):
    t = w.voronoi_tiling(N, L, seed)
    assert t.V == 2 * N
    h.check_topology(t.cell_vertex_num, t.cell_vertices, t.vertex_neighbors, t.vertex_cell_neighbors)
    ap = h.polygon_areas_numpy(t.pos, t.cell_vertex_num, t.cell_vertices, t.Lx, t.Ly)
    assert (ap[:, 0] > 0).all(), "rows must be counter-clockwise"
    assert abs(ap[:, 0].sum() - L * L) <= 1e-12 * L * L
    assert t.cell_vertex_num.mean() == 6.0
    assert (t.pos >= 0).all() and (t.pos[:, 0] < t.Lx).all() and (t.pos[:, 1] < t.Ly).all()


def test_voronoi_vertices_are_circumcentres_bruteforce():
    """Each vertex is equidistant from its three cells' generators and no generator is closer."""
    N, L = 400, 20.0
    t = w.voronoi_tiling(N, L, 5)
    pts = t.points
    for v in range(t.V):
        d = pts - t.pos[v]
        d = np.hypot(h.min_image(d[:, 0], L), h.min_image(d[:, 1], L))
        three = np.sort(d[t.vertex_cell_neighbors[v]])
        assert three[2] - three[0] < 1e-9
        assert d.min() > three[0] - 1e-9
        assert set(np.argsort(d)[:3].tolist()) == set(t.vertex_cell_neighbors[v].tolist())


@pytest.mark.parametrize("N,L,seed", [(64, 8.0, 1), (4096, 64.0, 2)])
def test_voronoi_matches_scipy(N, L, seed):
    """Vertex set equals scipy.spatial.Voronoi of the 3x3-replicated points (library cross-check)."""
    from scipy.spatial import Voronoi, cKDTree
    t = w.voronoi_tiling(N, L, seed)
    pts = t.points
    shifts = [(i * L, j * L) for i in (-1, 0, 1) for j in (-1, 0, 1)]
    big = np.vstack([pts + np.array(s) for s in shifts])
    vor = Voronoi(big)
    vv = vor.vertices
    inside = (vv[:, 0] >= 0) & (vv[:, 0] < L) & (vv[:, 1] >= 0) & (vv[:, 1] < L)
    vv = vv[inside]
    assert vv.shape[0] == t.V
    tree = cKDTree(vv)
    dist, idx = tree.query(t.pos)
    assert dist.max() < 1e-8
    assert len(set(idx.tolist())) == t.V
    # cell areas against scipy's regions of the central copy (centre block = index 4 in shifts)
    ap = h.polygon_areas_numpy(t.pos, t.cell_vertex_num, t.cell_vertices, t.Lx, t.Ly)
    from scipy.spatial import ConvexHull
    for c in range(0, N, max(1, N // 64)):
        region = vor.regions[vor.point_region[4 * N + c]]
        assert -1 not in region
        hull = ConvexHull(vor.vertices[region])
        assert abs(hull.volume - ap[c, 0]) < 1e-9       # 2-D "volume" is the area
        assert abs(hull.area - ap[c, 1]) < 1e-9         # 2-D "area" is the perimeter
        assert len(region) == t.cell_vertex_num[c]


def test_voronoi_side_histogram_is_poisson_voronoi_like():
    t = w.voronoi_tiling(65536, 256.0, 3)
    hist = np.bincount(t.cell_vertex_num, minlength=17) / t.N
    # Poisson-Voronoi: p6 ~ 0.295, p5 ~ 0.26, p7 ~ 0.20, p3 ~ 0.011
    assert 0.28 < hist[6] < 0.31 and 0.24 < hist[5] < 0.28 and 0.18 < hist[7] < 0.22
    assert 0.008 < hist[3] < 0.014
    assert t.cell_vertex_num.max() <= 16


def test_voronoi_is_seeded_and_deterministic():
    a = w.voronoi_tiling(256, 16.0, 9)
    b = w.voronoi_tiling(256, 16.0, 9)
    c = w.voronoi_tiling(256, 16.0, 10)
    assert np.array_equal(a.pos, b.pos) and np.array_equal(a.cell_vertices, b.cell_vertices)
    assert not np.array_equal(a.pos, c.pos)
    assert (a.theta >= 0).all() and (a.theta < 2 * np.pi).all()


def test_hex_tiling():
    t = w.hex_tiling(6, 4, a=0.7)
    h.check_topology(t.cell_vertex_num, t.cell_vertices, t.vertex_neighbors, t.vertex_cell_neighbors)
    ap = h.polygon_areas_numpy(t.pos, t.cell_vertex_num, t.cell_vertices, t.Lx, t.Ly)
    assert np.allclose(ap[:, 0], 1.5 * np.sqrt(3.0) * 0.49, rtol=1e-13)
    assert np.allclose(ap[:, 1], 6 * 0.7, rtol=1e-13)


def test_stride_overflow_is_reported():
    with pytest.raises(ValueError):
        w.voronoi_tiling(4096, 64.0, 2, S=8)
