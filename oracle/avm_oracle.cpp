// avm_oracle.cpp — CPU ORACLE for the active vertex model (AVM) hot path.  TEST INFRASTRUCTURE.
//
// A plain, slow, single-threaded, double-precision restatement of one overdamped AVM timestep
// as the paper defines it (arXiv:1702.02939, /root/reference/PAPER.md), following the algorithm
// step by step in the paper's order and notation.  Where the paper is silent the reading taken is
// the R-number of DESIGN.md §"Readings of the paper".
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// build, load or call this file.  It shares no code with the CUDA path (own Philox, own
// geometry, own T1) and imports nothing from paper_1702_02939_b200/.
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off -shared -fPIC (see oracle/__init__.py).  No
// -ffast-math: results must be reproducible across hosts (R21).
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`): regular-hexagon closed forms and zero force;
// forces vs central finite differences of Eq. A1; sum of areas = Lx*Ly; sum of forces = 0;
// shift invariance; Euler characteristic / 3-coordination / slot convention after T1 passes;
// hand-built T1 (Fig. 1 right); brute-force conflict rule; closed-form pure-activity translation;
// Philox core vs the cuRAND *host* generator (library routine) and moment/KS tests; per-cell targets and
// moduli vs finite differences of Eq. 1; mean-square displacement vs the closed-form translation, the
// closed form of one T1 and an independent numpy unwrapping of the trajectory.
// "Whole step" parity is unpinned beyond those invariants: the paper prints no trajectory.

#include <cstdint>
#include <cmath>
#include <cstring>
#include <vector>
#include <algorithm>
#include <utility>

namespace {

struct Params {
  int32_t n_cells, n_vertices, max_cell_vertices;
  int32_t t1_max_passes;   // NEXT-1: T1 passes per step; <= 1 = one pass (north_star), P > 1 = repeat until a
                           // pass finds no candidate, at most P passes
  double Lx, Ly;
  double KA, KP, A0, P0;      // Eq. A1: uniform moduli and preferred values (R17)
  double v0, Dr, mu, dt, l_c;
  uint64_t seed, step0;
};

struct Stats {
  int64_t step, t1_short, t1_candidates, t1_flips, t1_blocked, overflow_rejects, error;
};

struct Sim {
  Params p;
  int64_t N, V, S;
  std::vector<double> pos;      // [V][2]
  std::vector<double> theta;    // [N]
  std::vector<int32_t> cvn;     // [N]           cellVertexNum
  std::vector<int32_t> cv;      // [N][S]        cellVertices, counter-clockwise
  std::vector<int32_t> vn;      // [V][3]        vertexNeighbors
  std::vector<int32_t> vc;      // [V][3]        vertexCellNeighbors
  std::vector<double> A0c, P0c; // [N] per-cell preferred values A_{0,i}, P_{0,i} of Eq. 1 (
                                // NEXT-4); empty = the uniform A0, P0 of Eq. A1 (R17)
  std::vector<double> KAc, KPc; // [N] per-cell moduli K_{A,i}, K_{P,i} (Eq. 1 read with the moduli inside the sum,
                                // SURVEY 8(f) NEXT-4); empty = the uniform K_A, K_P of Eq. A1
  std::vector<double> unwrapped;  // [V][2] unwrapped positions: every elementary displacement (the Euler move of
                                  // Eq. 4, the repositioning of a T1) is added as a minimum-image vector, never wrapped
  std::vector<double> msd_ref;    // [V][2] unwrapped positions at the reference time of the mean-square displacement
  Stats st;
  double A0(int64_t c) const { return A0c.empty() ? p.A0 : A0c[c]; }
  double P0(int64_t c) const { return P0c.empty() ? p.P0 : P0c[c]; }
  double KA(int64_t c) const { return KAc.empty() ? p.KA : KAc[c]; }
  double KP(int64_t c) const { return KPc.empty() ? p.KP : KPc[c]; }
};

// ------------------------------------------------------------------------------------------
// Periodic box helpers (R13).  Positions stay in [0,L), so one correction suffices.
// ------------------------------------------------------------------------------------------
inline double mi(double d, double L) {
  if (d > 0.5 * L) d -= L;
  else if (d < -0.5 * L) d += L;
  return d;
}
inline double wrap(double x, double L) {
  if (x < 0.0) x += L;
  if (x >= L) x -= L;
  return x;
}

// ------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), R16.  ctr = 128-bit counter, key = 64 bit.
// ------------------------------------------------------------------------------------------
void philox4x32_10(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4]) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;   // round multipliers
  const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;   // key increments (Weyl sequence)
  uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3];
  uint32_t k0 = key_in[0], k1 = key_in[1];
  for (int r = 0; r < 10; ++r) {
    uint64_t p0 = (uint64_t)M0 * c0, p1 = (uint64_t)M1 * c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += W0; k1 += W1;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Standard normal for (seed, step, cell), R16: key = seed, counter = (step lo, step hi, cell lo,
// cell hi); two 52-bit uniforms in (0,1); Box-Muller cosine branch.
double director_noise(uint64_t seed, uint64_t step, uint64_t cell) {
  uint32_t ctr[4] = {(uint32_t)step, (uint32_t)(step >> 32), (uint32_t)cell, (uint32_t)(cell >> 32)};
  uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  uint32_t x[4];
  philox4x32_10(ctr, key, x);
  uint64_t a = ((uint64_t)x[1] << 32) | x[0], b = ((uint64_t)x[3] << 32) | x[2];
  const double two_m52 = 1.0 / 4503599627370496.0;
  double u1 = ((double)(a >> 12) + 0.5) * two_m52;
  double u2 = ((double)(b >> 12) + 0.5) * two_m52;
  return std::sqrt(-2.0 * std::log(u1)) * std::cos(6.283185307179586476925286766559 * u2);
}

// ------------------------------------------------------------------------------------------
// Step 1 — geometry of every cell ("the area and perimeter of every cell must first
// be computed"; :82 one unit of work per cell).  Shoelace sum over the CCW vertex list, every
// vertex unwrapped by minimum image relative to the row's first vertex (R14).  Areas are signed.
// ------------------------------------------------------------------------------------------
void cell_geometry(const Sim& s, int64_t c, double& A, double& P) {
  const int n = s.cvn[c];
  const int32_t* row = &s.cv[c * s.S];
  const double x0 = s.pos[2 * row[0]], y0 = s.pos[2 * row[0] + 1];
  std::vector<double> rx(n), ry(n);
  for (int j = 0; j < n; ++j) {
    rx[j] = mi(s.pos[2 * row[j]] - x0, s.p.Lx);
    ry[j] = mi(s.pos[2 * row[j] + 1] - y0, s.p.Ly);
  }
  A = 0.0; P = 0.0;
  for (int j = 0; j < n; ++j) {
    int jn = (j + 1) % n;
    A += rx[j] * ry[jn] - ry[j] * rx[jn];
    double dx = rx[jn] - rx[j], dy = ry[jn] - ry[j];
    P += std::sqrt(dx * dx + dy * dy);
  }
  A *= 0.5;
}

void geometry(const Sim& s, std::vector<double>& AP) {
  AP.resize(2 * s.N);
  for (int64_t c = 0; c < s.N; ++c) cell_geometry(s, c, AP[2 * c], AP[2 * c + 1]);
}

// Eq. 1 / A1: E = sum_i K_A (A_i - A0_i)^2 + K_P (P_i - P0_i)^2, no 1/2 (R4).
double energy(const Sim& s, const std::vector<double>& AP) {
  double E = 0.0;
  for (int64_t c = 0; c < s.N; ++c) {
    double dA = AP[2 * c] - s.A0(c), dP = AP[2 * c + 1] - s.P0(c);
    E += s.KA(c) * dA * dA + s.KP(c) * dP * dP;
  }
  return E;
}

// ------------------------------------------------------------------------------------------
// Step 2 — force on every vertex, Eq. A2-A5, F = -dE/dh (R1).
// For each of the three cells c bordering v ("the motion of vertex h_ijk only
// changes the shape of cells i, j, and k"):
//   dE_c/dh_v = 2 K_A (A_c-A0) dA_c/dh_v + 2 K_P (P_c-P0) dP_c/dh_v                 (A3)
//   dA_c/dh_v = 1/2 (r_next.y - r_prev.y, r_prev.x - r_next.x)                       (A4, R3)
//   dP_c/dh_v = -(rhat_prev + rhat_next), both unit vectors pointing away from v     (A5, R2)
// prev/next = v's neighbours in c's CCW row, found by searching the row (the definition; it
// does not rely on the slot convention).  A zero-length edge contributes 0 (R15).
// ------------------------------------------------------------------------------------------
void vertex_force(const Sim& s, const std::vector<double>& AP, int64_t v, double& Fx, double& Fy) {
  Fx = 0.0; Fy = 0.0;
  const double hx = s.pos[2 * v], hy = s.pos[2 * v + 1];
  for (int k = 0; k < 3; ++k) {
    const int64_t c = s.vc[3 * v + k];
    const int n = s.cvn[c];
    const int32_t* row = &s.cv[c * s.S];
    int j = -1;
    for (int t = 0; t < n; ++t) if (row[t] == v) { j = t; break; }
    const int32_t vp = row[(j + n - 1) % n], vx = row[(j + 1) % n];
    const double rpx = mi(s.pos[2 * vp] - hx, s.p.Lx), rpy = mi(s.pos[2 * vp + 1] - hy, s.p.Ly);
    const double rnx = mi(s.pos[2 * vx] - hx, s.p.Lx), rny = mi(s.pos[2 * vx + 1] - hy, s.p.Ly);
    const double dAx = 0.5 * (rny - rpy), dAy = 0.5 * (rpx - rnx);
    const double lp = std::sqrt(rpx * rpx + rpy * rpy), ln = std::sqrt(rnx * rnx + rny * rny);
    double upx = 0, upy = 0, unx = 0, uny = 0;
    if (lp > 0.0) { upx = rpx / lp; upy = rpy / lp; }
    if (ln > 0.0) { unx = rnx / ln; uny = rny / ln; }
    const double dPx = -(upx + unx), dPy = -(upy + uny);
    const double ca = 2.0 * s.KA(c) * (AP[2 * c] - s.A0(c)), cp = 2.0 * s.KP(c) * (AP[2 * c + 1] - s.P0(c));
    Fx -= ca * dAx + cp * dPx;
    Fy -= ca * dAy + cp * dPy;
  }
}

// ------------------------------------------------------------------------------------------
// Step 5 — one T1 pass (Fig. 1 right :27; R9-R12).
// ------------------------------------------------------------------------------------------
struct Cand {
  int32_t v1, v2;          // v1 < v2 (tags; the oracle never re-orders so tag == index)
  int k1, k2;              // slot of v2 in v1, slot of v1 in v2
  int32_t cL, cR, cE1, cE2;
};

// Short edges, eligibility (R10), in ascending key order (v1, v2).
// count: the pass adds to the t1_short / overflow_rejects statistics; raise: it may set the sticky
// error bit (the debug hook does neither)
void t1_candidates(Sim& s, std::vector<Cand>& cands, bool count, bool raise) {
  cands.clear();
  const double lc = s.p.l_c;
  for (int32_t v = 0; v < (int32_t)s.V; ++v) {
    // edges owned by the endpoint with the smaller tag; sort this vertex's partners so that the
    // list comes out in ascending (v1, v2)
    int order[3] = {0, 1, 2};
    std::sort(order, order + 3, [&](int a, int b) { return s.vn[3 * v + a] < s.vn[3 * v + b]; });
    for (int oi = 0; oi < 3; ++oi) {
      const int k = order[oi];
      const int32_t w = s.vn[3 * v + k];
      if (!(v < w)) continue;
      const double dx = mi(s.pos[2 * w] - s.pos[2 * v], s.p.Lx);
      const double dy = mi(s.pos[2 * w + 1] - s.pos[2 * v + 1], s.p.Ly);
      const double l = std::sqrt(dx * dx + dy * dy);
      if (!(l < lc)) continue;                       // strict (R9)
      if (count) ++s.st.t1_short;
      int k2 = -1;
      for (int t = 0; t < 3; ++t) if (s.vn[3 * w + t] == v) k2 = t;
      Cand c;
      c.v1 = v; c.v2 = w; c.k1 = k; c.k2 = k2;
      // slot convention (R12): cyclic from the partner's slot the cells are (C0, C1, C2);
      // C0 lies to the left of the directed edge u -> partner.
      c.cL = s.vc[3 * v + k];               // C0(v1): shares the edge, loses v1
      c.cE1 = s.vc[3 * v + (k + 1) % 3];    // C1(v1): end cell at v1, gains v2
      c.cR = s.vc[3 * w + k2];              // C0(v2): shares the edge, loses v2
      c.cE2 = s.vc[3 * w + (k2 + 1) % 3];   // C1(v2): end cell at v2, gains v1
      const bool distinct = c.cL != c.cR && c.cL != c.cE1 && c.cL != c.cE2 && c.cR != c.cE1 &&
                            c.cR != c.cE2 && c.cE1 != c.cE2;
      if (!distinct) continue;
      if (!(s.cvn[c.cL] > 3 && s.cvn[c.cR] > 3)) continue;          // no 2-gons; T2 not implemented
      if (!(s.cvn[c.cE1] < s.S && s.cvn[c.cE2] < s.S)) {            // row would exceed the stride
        // error bit 2 = "a flip was suppressed because a row would exceed S": raised whenever a
        // pass sees it (a repeated pass can be the first to see it, when an earlier pass of the
        // same step filled the end cell); the counter is a statistic of the step's first pass
        if (count) ++s.st.overflow_rejects;
        if (raise) s.st.error |= 2;
        continue;
      }
      cands.push_back(c);
    }
  }
}

inline uint64_t edge_key(const Cand& c) { return ((uint64_t)(uint32_t)c.v1 << 32) | (uint32_t)c.v2; }

// Conflict rule (R11; "a single topology update per cell per kernel call"): a
// candidate flips iff its key is the smallest among all candidates touching any of its 4 cells.
void t1_winners(const Sim& s, const std::vector<Cand>& cands, std::vector<char>& win) {
  std::vector<uint64_t> cellmin(s.N, ~0ull);
  for (const Cand& c : cands) {
    const uint64_t key = edge_key(c);
    for (int32_t cell : {c.cL, c.cR, c.cE1, c.cE2}) cellmin[cell] = std::min(cellmin[cell], key);
  }
  win.assign(cands.size(), 0);
  for (size_t i = 0; i < cands.size(); ++i) {
    const Cand& c = cands[i];
    const uint64_t key = edge_key(c);
    win[i] = cellmin[c.cL] == key && cellmin[c.cR] == key && cellmin[c.cE1] == key && cellmin[c.cE2] == key;
  }
}

void row_delete(Sim& s, int32_t c, int32_t v) {
  int32_t* row = &s.cv[(int64_t)c * s.S];
  int n = s.cvn[c], j = -1;
  for (int t = 0; t < n; ++t) if (row[t] == v) { j = t; break; }
  for (int t = j; t + 1 < n; ++t) row[t] = row[t + 1];
  row[n - 1] = -1;
  s.cvn[c] = n - 1;
}
void row_insert_after(Sim& s, int32_t c, int32_t after, int32_t v) {
  int32_t* row = &s.cv[(int64_t)c * s.S];
  int n = s.cvn[c], j = -1;
  for (int t = 0; t < n; ++t) if (row[t] == after) { j = t; break; }
  for (int t = n; t > j + 1; --t) row[t] = row[t - 1];
  row[j + 1] = v;
  s.cvn[c] = n + 1;
}

// One flip (R9 geometry, R12 rewrite).  Fig. 1 (right): cells i,k (here cL,cR) adjacent before,
// cells j,l (here cE1,cE2) adjacent after.
void t1_flip(Sim& s, const Cand& c) {
  const int32_t v1 = c.v1, v2 = c.v2;
  // --- geometry: rigid counter-clockwise quarter turn about the midpoint, new length 1.5 l_c
  const double h1x = s.pos[2 * v1], h1y = s.pos[2 * v1 + 1];
  const double dx = mi(s.pos[2 * v2] - h1x, s.p.Lx), dy = mi(s.pos[2 * v2 + 1] - h1y, s.p.Ly);
  const double l = std::sqrt(dx * dx + dy * dy);
  const double mx = h1x + 0.5 * dx, my = h1y + 0.5 * dy;
  double px = 0.0, py = 1.0;
  if (l > 0.0) { px = -dy / l; py = dx / l; }
  const double half = 0.75 * s.p.l_c;
  const double o1x = s.pos[2 * v1], o1y = s.pos[2 * v1 + 1], o2x = s.pos[2 * v2], o2y = s.pos[2 * v2 + 1];
  s.pos[2 * v2] = wrap(mx + half * px, s.p.Lx); s.pos[2 * v2 + 1] = wrap(my + half * py, s.p.Ly);
  s.pos[2 * v1] = wrap(mx - half * px, s.p.Lx); s.pos[2 * v1 + 1] = wrap(my - half * py, s.p.Ly);
  // unwrapped positions follow by the minimum-image displacement of the repositioning
  s.unwrapped[2 * v1] += mi(s.pos[2 * v1] - o1x, s.p.Lx); s.unwrapped[2 * v1 + 1] += mi(s.pos[2 * v1 + 1] - o1y, s.p.Ly);
  s.unwrapped[2 * v2] += mi(s.pos[2 * v2] - o2x, s.p.Lx); s.unwrapped[2 * v2 + 1] += mi(s.pos[2 * v2 + 1] - o2y, s.p.Ly);
  // --- topology.  Cyclic from the partner's slot: u has (n; c) = ([w, x, y]; [C0, C1, C2]).
  const int k1 = c.k1, k2 = c.k2;
  const int32_t x1 = s.vn[3 * v1 + (k1 + 1) % 3], y1 = s.vn[3 * v1 + (k1 + 2) % 3];
  const int32_t x2 = s.vn[3 * v2 + (k2 + 1) % 3], y2 = s.vn[3 * v2 + (k2 + 2) % 3];
  const int32_t L = c.cL, R = c.cR, E1 = c.cE1, E2 = c.cE2;
  // new (n; c) of u = ([w, y, z]; [C1, C2, C']), z = partner's old x, C' = partner's old C1
  s.vn[3 * v1 + k1] = v2; s.vn[3 * v1 + (k1 + 1) % 3] = y1; s.vn[3 * v1 + (k1 + 2) % 3] = x2;
  s.vc[3 * v1 + k1] = E1; s.vc[3 * v1 + (k1 + 1) % 3] = R;  s.vc[3 * v1 + (k1 + 2) % 3] = E2;
  s.vn[3 * v2 + k2] = v1; s.vn[3 * v2 + (k2 + 1) % 3] = y2; s.vn[3 * v2 + (k2 + 2) % 3] = x1;
  s.vc[3 * v2 + k2] = E2; s.vc[3 * v2 + (k2 + 1) % 3] = L;  s.vc[3 * v2 + (k2 + 2) % 3] = E1;
  // outer vertices: x1 was joined to v1 and is now joined to v2 (same slot); x2 likewise
  for (int t = 0; t < 3; ++t) if (s.vn[3 * x1 + t] == v1) { s.vn[3 * x1 + t] = v2; break; }
  for (int t = 0; t < 3; ++t) if (s.vn[3 * x2 + t] == v2) { s.vn[3 * x2 + t] = v1; break; }
  // rows: the two cells that shared the edge lose a vertex, the two end cells gain one
  row_delete(s, L, v1);
  row_delete(s, R, v2);
  row_insert_after(s, E1, v1, v2);
  row_insert_after(s, E2, v2, v1);
}

// returns the number of candidates of the pass (0 = the topology is at a fixed point of the rule)
// count_detect: whether this pass adds to the t1_short / overflow_rejects counters.  Reading
// (DESIGN.md section 9): both are statistics of the detection on the moved positions, i.e. of the
// step's first pass; repeated passes re-see the same short-but-ineligible edges and
// would count them once per pass.  The sticky error bit 2 is not a statistic: any pass raises it.
size_t t1_pass(Sim& s, bool count_detect = true) {
  std::vector<Cand> cands;
  std::vector<char> win;
  t1_candidates(s, cands, count_detect, true);
  t1_winners(s, cands, win);
  s.st.t1_candidates += (int64_t)cands.size();
  for (size_t i = 0; i < cands.size(); ++i) {
    if (win[i]) { t1_flip(s, cands[i]); ++s.st.t1_flips; }
    else ++s.st.t1_blocked;
  }
  return cands.size();
}

// ------------------------------------------------------------------------------------------
// One timestep in the paper's order (R6): geometry -> forces -> move the
// vertices with the current directors (Eq. 4, :56; R5, R7) -> rotate the directors (:50, :104;
// R8) -> test/update the topology on the moved positions (:64, :106-108) -> s <- s+1.
// ------------------------------------------------------------------------------------------
// The first four stages: everything up to, and excluding, the topology update.  Split off so that a test can
// look at the moved tiling of a step before its T1 pass (what the CUDA path's observing geometry
// pass reduces); step() below is the two halves back to back.
void step_move_and_rotate(Sim& s) {
  std::vector<double> AP;
  geometry(s, AP);                                                   // 1
  std::vector<double> F(2 * s.V);
  for (int64_t v = 0; v < s.V; ++v) vertex_force(s, AP, v, F[2 * v], F[2 * v + 1]);   // 2
  for (int64_t v = 0; v < s.V; ++v) {                                // 3: Eq. 4 with n = 3
    double ax = 0.0, ay = 0.0;
    for (int k = 0; k < 3; ++k) {
      const double th = s.theta[s.vc[3 * v + k]];
      ax += std::cos(th); ay += std::sin(th);
    }
    const double vx = s.p.mu * F[2 * v] + (s.p.v0 / 3.0) * ax;
    const double vy = s.p.mu * F[2 * v + 1] + (s.p.v0 / 3.0) * ay;
    s.unwrapped[2 * v] += s.p.dt * vx;                  // the displacement itself, before any wrap
    s.unwrapped[2 * v + 1] += s.p.dt * vy;
    s.pos[2 * v] = wrap(s.pos[2 * v] + s.p.dt * vx, s.p.Lx);
    s.pos[2 * v + 1] = wrap(s.pos[2 * v + 1] + s.p.dt * vy, s.p.Ly);
    if (!std::isfinite(s.pos[2 * v]) || !std::isfinite(s.pos[2 * v + 1])) s.st.error |= 1;
  }
  const double amp = std::sqrt(2.0 * s.p.Dr * s.p.dt);               // 4: Euler-Maruyama (R8)
  for (int64_t c = 0; c < s.N; ++c)
    s.theta[c] += amp * director_noise(s.p.seed, (uint64_t)s.st.step, (uint64_t)c);
}
void step_topology_and_advance(Sim& s) {
  // 5: one pass (north_star), or the paper's rule ("called repeatedly until no
  // changes"): repeat until a pass finds no candidate, at most t1_max_passes passes
  const int passes = s.p.t1_max_passes > 1 ? s.p.t1_max_passes : 1;
  for (int pass = 0; pass < passes; ++pass)
    if (t1_pass(s, pass == 0) == 0) break;
  ++s.st.step;                                                       // 6
}
void step(Sim& s) {
  step_move_and_rotate(s);
  step_topology_and_advance(s);
}

}  // namespace

// ==========================================================================================
// C entry points (host pointers only), loaded with ctypes by oracle/__init__.py
// ==========================================================================================
extern "C" {

typedef Params oracle_params;
typedef Stats oracle_stats;
typedef Sim oracle_sim;

oracle_sim* oracle_create(const oracle_params* p, const double* pos_xy, const int32_t* cell_vertex_num,
                          const int32_t* cell_vertices, const int32_t* vertex_neighbors,
                          const int32_t* vertex_cell_neighbors, const double* theta) {
  if (!p || p->n_cells <= 0 || p->n_vertices != 2 * p->n_cells || p->max_cell_vertices < 3) return nullptr;
  Sim* s = new Sim();
  s->p = *p;
  s->N = p->n_cells; s->V = p->n_vertices; s->S = p->max_cell_vertices;
  s->pos.assign(pos_xy, pos_xy + 2 * s->V);
  s->unwrapped = s->pos;
  s->msd_ref = s->pos;
  s->theta.assign(theta, theta + s->N);
  s->cvn.assign(cell_vertex_num, cell_vertex_num + s->N);
  s->cv.assign(cell_vertices, cell_vertices + s->N * s->S);
  s->vn.assign(vertex_neighbors, vertex_neighbors + 3 * s->V);
  s->vc.assign(vertex_cell_neighbors, vertex_cell_neighbors + 3 * s->V);
  std::memset(&s->st, 0, sizeof(Stats));
  s->st.step = (int64_t)p->step0;
  for (int64_t c = 0; c < s->N; ++c)
    if (s->cvn[c] < 3 || s->cvn[c] > s->S) { delete s; return nullptr; }
  return s;
}

void oracle_destroy(oracle_sim* s) { delete s; }

int oracle_geometry(oracle_sim* s, double* area_perim) {
  std::vector<double> AP;
  geometry(*s, AP);
  std::memcpy(area_perim, AP.data(), sizeof(double) * 2 * s->N);
  return 0;
}

double oracle_energy(oracle_sim* s) {
  std::vector<double> AP;
  geometry(*s, AP);
  return energy(*s, AP);
}

// = steps 1-2 on the current state, nothing modified (App. A.1)
int oracle_compute_forces(oracle_sim* s, double* force_xy, double* area_perim) {
  std::vector<double> AP;
  geometry(*s, AP);
  if (force_xy)
    for (int64_t v = 0; v < s->V; ++v) vertex_force(*s, AP, v, force_xy[2 * v], force_xy[2 * v + 1]);
  if (area_perim) std::memcpy(area_perim, AP.data(), sizeof(double) * 2 * s->N);
  return 0;
}

int oracle_step(oracle_sim* s, int64_t n_steps) {
  for (int64_t i = 0; i < n_steps; ++i) step(*s);
  return 0;
}
// the two halves of one step (test hooks): stages 1-4, then the topology update and the step counter
int oracle_step_move_and_rotate(oracle_sim* s) { step_move_and_rotate(*s); return 0; }
int oracle_step_topology_and_advance(oracle_sim* s) { step_topology_and_advance(*s); return 0; }

// one T1 pass on the current state without moving anything else (test hook)
// NEXT-4: per-cell preferred values of Eq. 1, user order; NULL, NULL = uniform again
int oracle_set_cell_targets(oracle_sim* s, const double* A0, const double* P0) {
  if (!s || ((A0 == nullptr) != (P0 == nullptr))) return -1;
  s->A0c.clear(); s->P0c.clear();
  if (A0) { s->A0c.assign(A0, A0 + s->N); s->P0c.assign(P0, P0 + s->N); }
  return 0;
}

// NEXT-4: per-cell moduli K_{A,i}, K_{P,i} (Eq. 1 with the moduli inside the sum), user order; NULL, NULL = uniform again
int oracle_set_cell_moduli(oracle_sim* s, const double* KA, const double* KP) {
  if (!s || ((KA == nullptr) != (KP == nullptr))) return -1;
  s->KAc.clear(); s->KPc.clear();
  if (KA) { s->KAc.assign(KA, KA + s->N); s->KPc.assign(KP, KP + s->N); }
  return 0;
}

// NEXT-2: mean-square displacement of the vertices since the reference time (creation, or the latest
// oracle_msd_reset): <|U_v(t) - U_v(t_ref)|^2> over all vertices, U = unwrapped position
double oracle_msd(oracle_sim* s) {
  double acc = 0.0;
  for (int64_t v = 0; v < s->V; ++v) {
    const double dx = s->unwrapped[2 * v] - s->msd_ref[2 * v], dy = s->unwrapped[2 * v + 1] - s->msd_ref[2 * v + 1];
    acc += dx * dx + dy * dy;
  }
  return acc / (double)s->V;
}
int oracle_msd_reset(oracle_sim* s) { s->msd_ref = s->unwrapped; return 0; }

int oracle_t1_pass(oracle_sim* s) { t1_pass(*s); return 0; }

// detect + resolve on the current state without flipping: sorted (tag_min, tag_max) pairs
int oracle_debug_t1(oracle_sim* s, int32_t* cand_pairs, int64_t* n_cand, int32_t* winner_pairs,
                    int64_t* n_win, int64_t capacity) {
  std::vector<Cand> cands;
  std::vector<char> win;
  t1_candidates(*s, cands, false, false);
  t1_winners(*s, cands, win);
  int64_t nc = 0, nw = 0;
  for (size_t i = 0; i < cands.size(); ++i) {
    if (nc < capacity && cand_pairs) { cand_pairs[2 * nc] = cands[i].v1; cand_pairs[2 * nc + 1] = cands[i].v2; }
    ++nc;
    if (win[i]) {
      if (nw < capacity && winner_pairs) { winner_pairs[2 * nw] = cands[i].v1; winner_pairs[2 * nw + 1] = cands[i].v2; }
      ++nw;
    }
  }
  *n_cand = nc; *n_win = nw;
  return 0;
}

int oracle_get_state(oracle_sim* s, double* pos_xy, int32_t* cell_vertex_num, int32_t* cell_vertices,
                     int32_t* vertex_neighbors, int32_t* vertex_cell_neighbors, double* theta,
                     oracle_stats* stats) {
  if (pos_xy) std::memcpy(pos_xy, s->pos.data(), sizeof(double) * 2 * s->V);
  if (cell_vertex_num) std::memcpy(cell_vertex_num, s->cvn.data(), sizeof(int32_t) * s->N);
  if (cell_vertices) std::memcpy(cell_vertices, s->cv.data(), sizeof(int32_t) * s->N * s->S);
  if (vertex_neighbors) std::memcpy(vertex_neighbors, s->vn.data(), sizeof(int32_t) * 3 * s->V);
  if (vertex_cell_neighbors) std::memcpy(vertex_cell_neighbors, s->vc.data(), sizeof(int32_t) * 3 * s->V);
  if (theta) std::memcpy(theta, s->theta.data(), sizeof(double) * s->N);
  if (stats) *stats = s->st;
  return 0;
}

// test hook: overwrite the positions; the unwrapped positions and the MSD reference restart from them
int oracle_set_positions(oracle_sim* s, const double* pos_xy) {
  std::memcpy(s->pos.data(), pos_xy, sizeof(double) * 2 * s->V);
  s->unwrapped = s->pos;
  s->msd_ref = s->pos;
  return 0;
}

void oracle_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox4x32_10(ctr, key, out); }

// raw words for (seed, step, cell0+i) with the counter/key layout of R16: out[4*i .. 4*i+3]
void oracle_philox_words(uint64_t seed, uint64_t step, uint64_t cell0, int64_t n, uint32_t* out) {
  for (int64_t i = 0; i < n; ++i) {
    uint64_t cell = cell0 + (uint64_t)i;
    uint32_t ctr[4] = {(uint32_t)step, (uint32_t)(step >> 32), (uint32_t)cell, (uint32_t)(cell >> 32)};
    uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    philox4x32_10(ctr, key, out + 4 * i);
  }
}

void oracle_director_noise(uint64_t seed, uint64_t step, uint64_t cell0, int64_t n, double* out) {
  for (int64_t i = 0; i < n; ++i) out[i] = director_noise(seed, step, cell0 + (uint64_t)i);
}

}  // extern "C"
