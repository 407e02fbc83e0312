"""Independent checkers used by the tests (numpy only; no oracle or CUDA code is called here).

* ``canonical_topology``  — the comparison form of DESIGN.md R19.
* ``check_topology``      — the invariants a 3-coordinated tiling on the torus must satisfy.
* ``polygon_areas_numpy`` — an independent shoelace over unwrapped polygons.
"""
from __future__ import annotations

import numpy as np


def min_image(d, L):
    return d - L * np.round(d / L)


def canonical_topology(cvn, cv, vn, vc):
    """R19: each vertex's (neighbour, cell) slot pairs rotated so that the smallest neighbour is
    first; each cell row rotated so that its smallest vertex is first (padding = -1)."""
    vn = np.asarray(vn)
    vc = np.asarray(vc)
    cv = np.asarray(cv)
    cvn = np.asarray(cvn)
    V = vn.shape[0]
    k = np.argmin(vn, axis=1)
    idx = (k[:, None] + np.arange(3)[None, :]) % 3
    vn_c = np.take_along_axis(vn, idx, axis=1)
    vc_c = np.take_along_axis(vc, idx, axis=1)
    N, S = cv.shape
    rows = np.full((N, S), -1, dtype=np.int64)
    big = np.where(np.arange(S)[None, :] < cvn[:, None], cv, np.iinfo(np.int32).max)
    k0 = np.argmin(big, axis=1)
    j = np.arange(S)[None, :]
    src = (k0[:, None] + j) % np.maximum(cvn[:, None], 1)
    rolled = np.take_along_axis(cv, src, axis=1)
    rows = np.where(j < cvn[:, None], rolled, -1)
    return dict(cvn=cvn.astype(np.int64), rows=rows, vn=vn_c.astype(np.int64), vc=vc_c.astype(np.int64))


def assert_same_topology(a, b):
    ca = canonical_topology(a["cell_vertex_num"], a["cell_vertices"], a["vertex_neighbors"], a["vertex_cell_neighbors"])
    cb = canonical_topology(b["cell_vertex_num"], b["cell_vertices"], b["vertex_neighbors"], b["vertex_cell_neighbors"])
    for key in ("cvn", "rows", "vn", "vc"):
        assert np.array_equal(ca[key], cb[key]), f"topology differs in {key}"


def check_topology(cvn, cv, vn, vc, S=None):
    """Invariants after any number of T1 passes (SURVEY §8(c) pins, T1 row)."""
    cvn = np.asarray(cvn)
    cv = np.asarray(cv)
    vn = np.asarray(vn)
    vc = np.asarray(vc)
    N, stride = cv.shape
    V = vn.shape[0]
    assert V == 2 * N
    assert cvn.min() >= 3 and cvn.max() <= stride
    assert int(cvn.sum()) == 6 * N, "sum of cellVertexNum must be 6N"
    # Euler characteristic of the torus: V - E + F = 0 with E = 3V/2
    n_edges = sum(1 for v in range(V) for w in vn[v] if v < w)
    assert V - n_edges + N == 0
    # three distinct neighbours / cells, symmetric neighbour relation
    for v in range(V):
        assert len(set(vn[v].tolist())) == 3 and v not in vn[v], f"vertex {v} neighbours {vn[v]}"
        assert len(set(vc[v].tolist())) == 3, f"vertex {v} cells {vc[v]}"
        for w in vn[v]:
            assert v in vn[w], f"neighbour relation not symmetric at ({v},{w})"
    # padding and membership
    count = np.zeros(V, dtype=np.int64)
    for c in range(N):
        n = cvn[c]
        row = cv[c, :n]
        assert (cv[c, n:] == -1).all(), f"row {c} padding"
        assert len(set(row.tolist())) == n
        count[row] += 1
        for j in range(n):
            v, nxt, prv = row[j], row[(j + 1) % n], row[(j - 1) % n]
            # slot convention R12: for the slot k with vc[v][k] == c, next = vn[v][k], prev = vn[v][k+1]
            ks = [k for k in range(3) if vc[v][k] == c]
            assert len(ks) == 1, f"cell {c} not (uniquely) among cells of vertex {v}"
            k = ks[0]
            assert vn[v][k] == nxt and vn[v][(k + 1) % 3] == prv, f"slot convention broken at v={v}, c={c}"
    assert (count == 3).all(), "every vertex must appear in exactly three rows"


def unwrapped_polygons(pos, cvn, cv, Lx, Ly):
    """List of [n,2] arrays: each cell's vertices unwrapped by walking edge to edge."""
    polys = []
    for c in range(cv.shape[0]):
        n = cvn[c]
        p = pos[cv[c, :n]]
        d = np.diff(p, axis=0)
        d[:, 0] = min_image(d[:, 0], Lx)
        d[:, 1] = min_image(d[:, 1], Ly)
        q = np.vstack([np.zeros((1, 2)), np.cumsum(d, axis=0)]) + p[0]
        polys.append(q)
    return polys


def polygon_areas_numpy(pos, cvn, cv, Lx, Ly):
    out = np.empty((cv.shape[0], 2))
    for c, q in enumerate(unwrapped_polygons(pos, cvn, cv, Lx, Ly)):
        x, y = q[:, 0] - q[0, 0], q[:, 1] - q[0, 1]   # relative coordinates: less round-off
        out[c, 0] = 0.5 * np.sum(x * np.roll(y, -1) - y * np.roll(x, -1))
        e = np.roll(q, -1, axis=0) - q
        out[c, 1] = np.sum(np.hypot(e[:, 0], e[:, 1]))
    return out


def cells_adjacent(cv, cvn, a, b):
    """True if cells a and b share an edge (two consecutive common vertices)."""
    ra = cv[a, :cvn[a]].tolist()
    rb = set(cv[b, :cvn[b]].tolist())
    n = len(ra)
    return any(ra[j] in rb and ra[(j + 1) % n] in rb for j in range(n))
