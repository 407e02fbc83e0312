"""CPU oracle of the GPU-only parts of one self-propelled-Voronoi (SPV) step on a FIXED triangulation.

TEST INFRASTRUCTURE ONLY, like everything under ``oracle/``: plain numpy in float64, no blocking,
no fusion, written from the definitions so that it can be checked against the paper by eye.  It
shares no code with the CUDA path.  Only ``tests/`` may import it.

What the paper's SPV loop does on the GPU (PAPER.md:80-94, section II.C; App. A.2, :171-200) and what
this file restates:

  1. geometry  - the Voronoi vertex of every Delaunay triangle is the circumcentre of its three
                 cell positions; cell area and perimeter follow from the CCW list of those
                 vertices;
  2. forces    - F_i = -dE/dr_i with E of Eq. 1, decomposed into "force sets", the
                 contribution of each Voronoi vertex of cell i (Eq. A6-A7):
                     F_i = - sum over the vertices v of cell i of (dh_v/dr_i)^T dE/dh_v ,
                 where dE/dh_v is the vertex-model derivative of App. A.1 (the AVM oracle evaluates
                 it) and dh_v/dr_i is the derivative of a circumcentre with respect to one corner;
  3. move      - Eq. 3: dr_i/dt = mu F_i + v0 n_i, explicit Euler, then the director
                 noise of PAPER.md:50 (the same Philox-keyed Euler-Maruyama update as the AVM);
  4. test      - the empty-circumcircle property of every triangle.

The triangulation is the dual reading of the AVM's three lists: vertex v <-> triangle
with corners vertex_cell_neighbors[v]; row c of cell_vertices = the triangles around cell c, CCW;
vertex_neighbors[v] = the three adjacent triangles.  The CPU/CGAL repair of PAPER.md:96-100 is out of
scope on both sides.

Readings:
  S1  Eq. A11-A14 are garbled in PAPER.md (A12 prints r_ik . r_ik).  dh/dr_i is therefore taken from the
      definition: h = r_i + u(b, c), b = r_j - r_i, c = r_k - r_i,
          D = 2 (b_x c_y - b_y c_x),  u = ( c_y |b|^2 - b_y |c|^2 ,  b_x |c|^2 - c_x |b|^2 ) / D ,
      differentiated with the quotient rule (d b/d r_i = d c/d r_i = -1).  Pinned by central finite
      differences of E and of h.
  S2  which cells a triangle's circumcircle is tested against (paper: "to see if any cell has moved in
      such a way that an update ... is needed"): the cell opposite each of its three edges, i.e. the corner
      of the adjacent triangle that the triangle does not share.  A triangulation all of whose edges pass
      this local test is the Delaunay triangulation (the classical local-Delaunay lemma), so the verdict
      "valid / needs repair" equals that of the global test; `test_triangulation_global` is the global
      test by brute force, used by the pins.
  S3  strict test: a cell exactly on the circle does not fail.

parity: every function here is pinned in tests/test_oracle_spv.py (circumcentres of a Voronoi start
reproduce the generator's vertices; equidistance; forces against central differences of the energy,
zero on the triangular lattice, zero net force; Eq. 3 closed forms; local verdict == global verdict).
"""
from __future__ import annotations

import numpy as np

import oracle


def _mi(d, L):
    """minimum image of a difference, one correction (positions stay in [0, L))"""
    return d - L * np.rint(d / L)


class SpvOracle:
    def __init__(self, t, cell_xy, **params):
        self.t = t
        self.N, self.V, self.S = t.N, t.V, t.S
        self.L = np.array([t.Lx, t.Ly])
        self.p = dict(KA=1.0, KP=1.0, A0=1.0, P0=3.8, v0=0.0, Dr=0.0, mu=1.0, dt=0.01, seed=0)
        self.p.update({k: v for k, v in params.items() if k in self.p})
        self.r = np.array(cell_xy, dtype=np.float64)
        self.theta = np.array(t.theta, dtype=np.float64)
        self.step_count = 0
        self.vc = t.vertex_cell_neighbors
        self.vn = t.vertex_neighbors

    # ---- 1. geometry ----
    def circumcentres(self, r=None):
        """h_v for every triangle, wrapped into the box; also b, c (the two edge vectors from corner 0)"""
        r = self.r if r is None else r
        r0 = r[self.vc[:, 0]]
        b = _mi(r[self.vc[:, 1]] - r0, self.L)
        c = _mi(r[self.vc[:, 2]] - r0, self.L)
        D = 2.0 * (b[:, 0] * c[:, 1] - b[:, 1] * c[:, 0])
        b2, c2 = (b * b).sum(1), (c * c).sum(1)
        u = np.stack([c[:, 1] * b2 - b[:, 1] * c2, b[:, 0] * c2 - c[:, 0] * b2], axis=1) / D[:, None]
        h = np.mod(r0 + u, self.L)
        h[h >= self.L] = 0.0                      # a tiny negative coordinate wraps to L in floating point
        return h

    def _avm(self, h):
        """the AVM oracle on the Voronoi vertices: areas, perimeters and dE/dh (App. A.1)"""
        t = self.t
        return oracle.OracleSim(h, t.cell_vertex_num, t.cell_vertices, t.vertex_neighbors, t.vertex_cell_neighbors,
                                self.theta, Lx=t.Lx, Ly=t.Ly, **{k: self.p[k] for k in ("KA", "KP", "A0", "P0")})

    def geometry(self, r=None):
        """(Voronoi vertices [V,2], (A_c, P_c) [N,2])"""
        h = self.circumcentres(r)
        return h, self._avm(h).geometry()

    def energy(self, r=None):
        """Eq. 1 of the tiling whose vertices are the circumcentres"""
        _, ap = self.geometry(r)
        return float((self.p["KA"] * (ap[:, 0] - self.p["A0"]) ** 2 + self.p["KP"] * (ap[:, 1] - self.p["P0"]) ** 2).sum())

    # ---- 2. forces (Eq. A6-A7; reading S1) ----
    def dh_dr(self, r=None):
        """J[v, k] = d h_v / d r_(corner k), a 2x2 matrix (row = component of h, column = component of r)"""
        r = self.r if r is None else r
        J = np.zeros((self.V, 3, 2, 2))
        for k in range(3):                      # the corner that moves plays the role of r_i; the other two are j, k
            ri = r[self.vc[:, k]]
            b = _mi(r[self.vc[:, (k + 1) % 3]] - ri, self.L)
            c = _mi(r[self.vc[:, (k + 2) % 3]] - ri, self.L)
            b2, c2 = (b * b).sum(1), (c * c).sum(1)
            D = 2.0 * (b[:, 0] * c[:, 1] - b[:, 1] * c[:, 0])
            nx = c[:, 1] * b2 - b[:, 1] * c2            # numerators of u
            ny = b[:, 0] * c2 - c[:, 0] * b2
            # partial derivatives with respect to (b_x, b_y, c_x, c_y)
            dD = np.stack([2.0 * c[:, 1], -2.0 * c[:, 0], -2.0 * b[:, 1], 2.0 * b[:, 0]], axis=1)
            dnx = np.stack([2.0 * c[:, 1] * b[:, 0], 2.0 * c[:, 1] * b[:, 1] - c2, -2.0 * b[:, 1] * c[:, 0], b2 - 2.0 * b[:, 1] * c[:, 1]], axis=1)
            dny = np.stack([c2 - 2.0 * c[:, 0] * b[:, 0], -2.0 * c[:, 0] * b[:, 1], 2.0 * b[:, 0] * c[:, 0] - b2, 2.0 * b[:, 0] * c[:, 1]], axis=1)
            dux = (dnx * D[:, None] - nx[:, None] * dD) / (D * D)[:, None]     # quotient rule
            duy = (dny * D[:, None] - ny[:, None] * dD) / (D * D)[:, None]
            # h = r_i + u(b, c), db/dr_i = dc/dr_i = -1:  dh/dr_i = 1 - du/db - du/dc
            J[:, k, 0, 0] = 1.0 - dux[:, 0] - dux[:, 2]
            J[:, k, 0, 1] = -dux[:, 1] - dux[:, 3]
            J[:, k, 1, 0] = -duy[:, 0] - duy[:, 2]
            J[:, k, 1, 1] = 1.0 - duy[:, 1] - duy[:, 3]
        return J

    def force_sets(self, r=None):
        """f[c, j] = force on cell c due to the j-th Voronoi vertex of its row, [N, S, 2]"""
        r = self.r if r is None else r
        h = self.circumcentres(r)
        Fv, _ = self._avm(h).compute_forces()          # F_v = -dE/dh_v (App. A.1)
        g = -Fv
        J = self.dh_dr(r)
        t = self.t
        f = np.zeros((self.N, self.S, 2))
        for c in range(self.N):
            for j in range(int(t.cell_vertex_num[c])):
                v = int(t.cell_vertices[c, j])
                k = int(np.nonzero(self.vc[v] == c)[0][0])
                f[c, j] = -J[v, k].T @ g[v]
        return f

    def forces(self, r=None):
        """F_i = sum of its force sets in row order (PAPER.md:88 second kernel)"""
        f = self.force_sets(r)
        F = np.zeros((self.N, 2))
        for j in range(self.S):
            F += f[:, j]
        return F

    # ---- 3. Eq. 3 + director noise ----
    def step(self, n=1):
        p = self.p
        amp = np.sqrt(2.0 * p["Dr"] * p["dt"])
        for _ in range(n):
            F = self.forces()
            nvec = np.stack([np.cos(self.theta), np.sin(self.theta)], axis=1)     # directors at the start of the step
            self.r = np.mod(self.r + p["dt"] * (p["mu"] * F + p["v0"] * nvec), self.L)
            self.r[self.r >= self.L] = 0.0
            self.theta = self.theta + amp * oracle.director_noise(p["seed"], self.step_count, 0, self.N)
            self.step_count += 1

    # ---- 4. empty-circumcircle test (readings S2, S3) ----
    def _circles(self, r):
        r0 = r[self.vc[:, 0]]
        b = _mi(r[self.vc[:, 1]] - r0, self.L)
        c = _mi(r[self.vc[:, 2]] - r0, self.L)
        D = 2.0 * (b[:, 0] * c[:, 1] - b[:, 1] * c[:, 0])
        b2, c2 = (b * b).sum(1), (c * c).sum(1)
        u = np.stack([c[:, 1] * b2 - b[:, 1] * c2, b[:, 0] * c2 - c[:, 0] * b2], axis=1) / D[:, None]
        return r0, u, (u * u).sum(1)             # corner 0, centre relative to it, radius^2

    def test_triangulation(self, r=None, band=0.0):
        """local test: (failed[v, k] for the cell opposite edge k of triangle v, margin (d^2 - R^2) / R^2)"""
        r = self.r if r is None else r
        r0, u, R2 = self._circles(r)
        failed = np.zeros((self.V, 3), dtype=bool)
        margin = np.zeros((self.V, 3))
        opp = np.zeros((self.V, 3), dtype=np.int64)
        for k in range(3):
            w = self.vn[:, k]
            for m in range(3):                   # the corner of the adjacent triangle that v does not share
                cand = self.vc[w, m]
                notmine = (cand != self.vc[:, 0]) & (cand != self.vc[:, 1]) & (cand != self.vc[:, 2])
                opp[notmine, k] = cand[notmine]
            d = _mi(r[opp[:, k]] - r0, self.L) - u
            d2 = (d * d).sum(1)
            margin[:, k] = (d2 - R2) / R2
            failed[:, k] = d2 < R2
        return failed, margin, opp

    def test_triangulation_global(self, r=None):
        """brute force: triangle v fails iff ANY cell other than its corners lies strictly inside its circle"""
        r = self.r if r is None else r
        r0, u, R2 = self._circles(r)
        bad = np.zeros(self.V, dtype=bool)
        for v in range(self.V):
            d = _mi(r - r0[v], self.L) - u[v]
            d2 = (d * d).sum(1)
            d2[self.vc[v]] = np.inf
            bad[v] = (d2 < R2[v] * (1.0 - 1e-12)).any()
        return bad
