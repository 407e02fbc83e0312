"""A valid 3-coordinated tiling of the torus in which ONE cell touches both ends of an edge it does not contain
(the end cells of that edge coincide: E1 == E2).  DESIGN.md R10 keeps such an edge from flipping ("the four cells
are distinct"); the pins of that clause (tests/test_oracle_t1.py, tests/test_gpu_parity.py) need a state that has one.

Three of the six inequalities of R10 hold in every valid tiling (a vertex has three distinct cells, so E1 != L, R
and E2 != L, R) and L != R holds for cells narrower than half the box; E1 == E2 is the case that remains: a cell
that wraps around a group of others.  No generator of this repository produces one, but T1s can: the state is
reached from the 4 x 4 hexagonal torus by a seeded sequence of T1 passes of the oracle on arbitrary positions
(topology only - forces play no role), scanning the lists after every pass.  The lists are then checked by the
independent checker tests/helpers.check_topology, so nothing about the oracle's flips is taken on trust."""
from __future__ import annotations

import types

import numpy as np

import oracle
from paper_1702_02939_b200 import workloads as w

PARAMS = dict(KA=0.0, KP=0.0, A0=1.0, P0=3.8, v0=0.0, Dr=0.0, mu=1.0, dt=0.0, l_c=0.3, seed=1)


def edges_whose_end_cells_coincide(vn, vc):
    """[(v1, v2, L, R, E)] with E = the cell after the partner's slot at both ends (slot convention R12)"""
    out = []
    for v in range(vn.shape[0]):
        for k in range(3):
            u = int(vn[v, k])
            if v > u:
                continue
            k2 = [t for t in range(3) if vn[u, t] == v][0]
            if vc[v, (k + 1) % 3] == vc[u, (k2 + 1) % 3]:
                out.append((v, u, int(vc[v, k]), int(vc[u, k2]), int(vc[v, (k + 1) % 3])))
    return out


def build(seed: int = 0):
    """(tiling-like namespace, (v1, v2, L, R, E)): positions put only the edge (v1, v2) below l_c = 0.3"""
    t = w.hex_tiling(4, 4, a=1.0)
    box = np.array([t.Lx, t.Ly])
    V = t.pos.shape[0]
    rng = np.random.default_rng(seed)
    o = oracle.from_tiling(t, **PARAMS)
    for _ in range(2000):
        st = o.get_state()
        pos = rng.random((V, 2)) * box
        for _ in range(2):                      # two random edges become short: the pass flips them
            v = int(rng.integers(V))
            u = int(st["vertex_neighbors"][v, rng.integers(3)])
            pos[u] = np.mod(pos[v] + 0.01 * rng.standard_normal(2), box)
        o.set_positions(pos)
        o.t1_pass()
        st = o.get_state()
        cvn = st["cell_vertex_num"]
        good = [e for e in edges_whose_end_cells_coincide(st["vertex_neighbors"], st["vertex_cell_neighbors"])
                if cvn[e[2]] > 3 and cvn[e[3]] > 3 and cvn[e[4]] < t.S - 1]      # every other clause of R10 lets it through
        if good:
            break
    else:
        raise AssertionError("no such state found")
    v1, v2 = good[0][:2]
    # positions: a jittered grid keeps every pair of vertices at least 0.5 apart; then v2 moves next to v1
    n = int(np.ceil(np.sqrt(V)))
    grid = np.stack(np.meshgrid(np.arange(n), np.arange(n), indexing="ij"), axis=-1).reshape(-1, 2)[:V]
    pos = (grid + 0.5) * (box / n) + 0.05 * (rng.random((V, 2)) - 0.5)
    assert (box / n).min() > 0.7
    pos[v2] = np.mod(pos[v1] + np.array([0.06, 0.03]), box)
    out = types.SimpleNamespace(N=t.N, S=t.S, Lx=t.Lx, Ly=t.Ly, pos=pos, cell_vertex_num=st["cell_vertex_num"].copy(),
                                cell_vertices=st["cell_vertices"].copy(), vertex_neighbors=st["vertex_neighbors"].copy(),
                                vertex_cell_neighbors=st["vertex_cell_neighbors"].copy(), theta=np.zeros(t.N))
    return out, good[0]
