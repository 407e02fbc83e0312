// tiling.cpp — seeded synthetic INPUT generator for the AVM hot path.
//
// Produces the initial state the BASELINE.json configs describe: "Voronoi of N uniform-random
// points (seed k)" in a periodic box, as the three flat topology lists of PAPER.md:66 (§II.B:
// vertices around each cell in counter-clockwise order, vertices each vertex is connected to,
// cells that border each vertex).  DESIGN.md §"Input recipe" states the construction.
//
// This module serves both the CPU oracle's tests and the CUDA path's tests/bench.  It contains
// none of the method's arithmetic (no area/perimeter/force/T1/integrator code, no Philox): it
// only builds a 3-coordinated periodic tiling and the index lists that describe it.  Its random
// numbers come from SplitMix64, a generator neither the oracle nor the CUDA path uses.
//
// Build: g++ -O2 -shared -fPIC -o libavm_tiling.so tiling.cpp   (see workloads/__init__.py)

#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <cmath>
#include <vector>
#include <algorithm>

namespace {

inline uint64_t splitmix64(uint64_t z) {
  z += 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
// counter-based uniform in [0,1): stream selects an independent sequence
inline double uniform01(uint64_t seed, uint64_t stream, uint64_t i) {
  uint64_t k = splitmix64(seed * 0x2545F4914F6CDD1Dull + stream);
  uint64_t r = splitmix64(k ^ splitmix64(i));
  return (double)(r >> 11) * (1.0 / 9007199254740992.0);
}

inline double min_image(double d, double L) {
  if (d > 0.5 * L) d -= L; else if (d < -0.5 * L) d += L;
  return d;
}
inline double wrap(double x, double L) {
  if (x < 0.0) x += L;
  if (x >= L) x -= L;
  return x;
}

constexpr int MAXP = 96;  // working polygon capacity during clipping

struct Poly {
  int n;
  double x[MAXP], y[MAXP];
  int nbr[MAXP];  // nbr[k] = point whose bisector carries the edge from vertex k to vertex k+1
};

// Clip convex polygon (relative to the generator at the origin) by the half-plane of points
// closer to the origin than to d=(dx,dy).  Returns false on overflow.
bool clip(Poly& P, double dx, double dy, int j) {
  const double h = 0.5 * (dx * dx + dy * dy);
  double s[MAXP];
  bool any_out = false, any_in = false;
  for (int k = 0; k < P.n; ++k) {
    s[k] = P.x[k] * dx + P.y[k] * dy - h;
    if (s[k] > 0.0) any_out = true; else any_in = true;
  }
  if (!any_out) return true;
  if (!any_in) return false;  // cannot happen: the origin is always inside
  // find first outside vertex whose predecessor is inside
  int n = P.n, first_out = -1;
  for (int k = 0; k < n; ++k) {
    int kp = (k + n - 1) % n;
    if (s[k] > 0.0 && s[kp] <= 0.0) { first_out = k; break; }
  }
  int last_out = first_out;
  while (s[(last_out + 1) % n] > 0.0) last_out = (last_out + 1) % n;
  int a = (first_out + n - 1) % n;  // last inside before the run
  int b = (last_out + 1) % n;       // first inside after the run
  // intersection on edge a -> first_out (keeps label nbr[a]) and on edge last_out -> b
  double ta = s[a] / (s[a] - s[first_out]);
  double Ax = P.x[a] + ta * (P.x[first_out] - P.x[a]);
  double Ay = P.y[a] + ta * (P.y[first_out] - P.y[a]);
  double tb = s[last_out] / (s[last_out] - s[b]);
  double Bx = P.x[last_out] + tb * (P.x[b] - P.x[last_out]);
  double By = P.y[last_out] + tb * (P.y[b] - P.y[last_out]);
  int lab_last = P.nbr[last_out];
  // rebuild: walk from b around to a (inside run), then A (edge label j), then B (label lab_last)
  Poly Q;
  Q.n = 0;
  for (int k = b;; k = (k + 1) % n) {
    Q.x[Q.n] = P.x[k]; Q.y[Q.n] = P.y[k]; Q.nbr[Q.n] = P.nbr[k]; ++Q.n;
    if (k == a) break;
  }
  if (Q.n + 2 > MAXP) return false;
  Q.x[Q.n] = Ax; Q.y[Q.n] = Ay; Q.nbr[Q.n] = j; ++Q.n;
  Q.x[Q.n] = Bx; Q.y[Q.n] = By; Q.nbr[Q.n] = lab_last; ++Q.n;
  P = Q;
  return true;
}

}  // namespace

extern "C" {

// error codes (negative)
enum {
  TILING_OK = 0,
  TILING_EBADARG = -1,
  TILING_EOPEN = -2,        // a cell stayed unbounded by neighbours (box too small for the search)
  TILING_ESTRIDE = -3,      // a cell has more than S vertices
  TILING_EMISMATCH = -4,    // a vertex triple was not produced exactly three times (degenerate input)
  TILING_ECOUNT = -5,       // V != 2N
  TILING_ECLIP = -6,
  TILING_ESLOT = -7         // rows do not describe a 3-coordinated tiling
};

// Uniform points in [0,Lx)x[0,Ly): point i = (u(seed,stream 1,i)*Lx, u(seed,stream 2,i)*Ly).
int tiling_points(int64_t N, double Lx, double Ly, uint64_t seed, double* pts_xy) {
  if (N <= 0 || !pts_xy) return TILING_EBADARG;
  for (int64_t i = 0; i < N; ++i) {
    pts_xy[2 * i] = uniform01(seed, 1, (uint64_t)i) * Lx;
    pts_xy[2 * i + 1] = uniform01(seed, 2, (uint64_t)i) * Ly;
  }
  return TILING_OK;
}

// Initial directors: theta_i uniform in [0, 2*pi), stream 3 of the same seed.
int tiling_thetas(int64_t N, uint64_t seed, double* theta) {
  if (N <= 0 || !theta) return TILING_EBADARG;
  for (int64_t i = 0; i < N; ++i) theta[i] = uniform01(seed, 3, (uint64_t)i) * 6.283185307179586476925286766559;
  return TILING_OK;
}

// Build vertexNeighbors / vertexCellNeighbors from CCW cell rows, in the slot convention of
// DESIGN.md (§Data layout): neighbours n0,n1,n2 counter-clockwise around v; cell c_k lies between
// edges (v,n_k) and (v,n_{k+1}), i.e. in c_k's row (n_{k+1}, v, n_k) are consecutive.
int tiling_from_rows(int64_t N, int64_t V, int32_t S, const int32_t* cvn, const int32_t* cv,
                     int32_t* vn, int32_t* vc) {
  if (N <= 0 || V <= 0 || S < 3) return TILING_EBADARG;
  std::vector<int32_t> cnt(V, 0);
  std::vector<int32_t> ec(3 * V), en(3 * V), ep(3 * V);  // per vertex entries: cell, next, prev
  for (int64_t c = 0; c < N; ++c) {
    int n = cvn[c];
    if (n < 3 || n > S) return TILING_ESTRIDE;
    const int32_t* row = cv + c * S;
    for (int k = 0; k < n; ++k) {
      int32_t v = row[k];
      if (v < 0 || v >= V) return TILING_ESLOT;
      if (cnt[v] >= 3) return TILING_ESLOT;
      int e = 3 * v + cnt[v]++;
      ec[e] = (int32_t)c;
      en[e] = row[(k + 1) % n];
      ep[e] = row[(k + n - 1) % n];
    }
  }
  for (int64_t v = 0; v < V; ++v) {
    if (cnt[v] != 3) return TILING_ESLOT;
    int e0 = 3 * v;
    int32_t n0 = en[e0], n1 = ep[e0];
    int e1 = -1, e2 = -1;
    for (int t = 1; t < 3; ++t) if (en[3 * v + t] == n1) e1 = 3 * v + t;
    if (e1 < 0) return TILING_ESLOT;
    int32_t n2 = ep[e1];
    for (int t = 1; t < 3; ++t) if (3 * v + t != e1 && en[3 * v + t] == n2) e2 = 3 * v + t;
    if (e2 < 0 || ep[e2] != n0) return TILING_ESLOT;
    vn[3 * v] = n0; vn[3 * v + 1] = n1; vn[3 * v + 2] = n2;
    vc[3 * v] = ec[e0]; vc[3 * v + 1] = ec[e1]; vc[3 * v + 2] = ec[e2];
  }
  return TILING_OK;
}

// Periodic Voronoi tiling of the given points.  Outputs:
//   pos_xy[2*2N]   vertex positions (circumcentres), wrapped into the box
//   cvn[N], cv[N*S] CCW rows (unused slots = -1); vn[3*2N], vc[3*2N] in the slot convention
//   info[0] = max vertices per cell, info[1] = number of vertices produced
// Vertex numbering: order of first appearance scanning cells 0..N-1, each row counter-clockwise
// from its first vertex (the vertex whose outgoing edge borders the smallest-index neighbour).
int tiling_voronoi(int64_t N, double Lx, double Ly, const double* pts, int32_t S, double* pos_xy,
                   int32_t* cvn, int32_t* cv, int32_t* vn, int32_t* vc, int64_t* info) {
  if (N < 4 || Lx <= 0 || Ly <= 0 || S < 3 || S > 64) return TILING_EBADARG;
  // uniform grid with about 2 points per grid cell
  const double area = Lx * Ly;
  double g0 = std::sqrt(2.0 * area / (double)N);
  int64_t Gx = std::max<int64_t>(1, (int64_t)std::floor(Lx / g0));
  int64_t Gy = std::max<int64_t>(1, (int64_t)std::floor(Ly / g0));
  const double gx = Lx / (double)Gx, gy = Ly / (double)Gy;
  const double g = std::min(gx, gy);
  std::vector<int64_t> start(Gx * Gy + 1, 0);
  std::vector<int32_t> items(N);
  auto cell_of = [&](int64_t i, int64_t& ix, int64_t& iy) {
    ix = (int64_t)std::floor(pts[2 * i] / gx); iy = (int64_t)std::floor(pts[2 * i + 1] / gy);
    if (ix >= Gx) ix = Gx - 1; if (iy >= Gy) iy = Gy - 1;
    if (ix < 0) ix = 0; if (iy < 0) iy = 0;
  };
  for (int64_t i = 0; i < N; ++i) { int64_t ix, iy; cell_of(i, ix, iy); ++start[iy * Gx + ix + 1]; }
  for (int64_t k = 0; k < Gx * Gy; ++k) start[k + 1] += start[k];
  {
    std::vector<int64_t> fill(start.begin(), start.end() - 1);
    for (int64_t i = 0; i < N; ++i) { int64_t ix, iy; cell_of(i, ix, iy); items[fill[iy * Gx + ix]++] = (int32_t)i; }
  }
  std::vector<int32_t> cnbr((size_t)N * S, -1);  // neighbour label of the edge leaving each row slot
  std::vector<uint8_t> seen;                      // times each vertex was produced
  seen.reserve(2 * N);
  int64_t V = 0, maxn = 0;
  const int64_t Rmax = std::max(Gx, Gy) / 2 + 1;
  for (int64_t c = 0; c < N * S; ++c) cv[c] = -1;

  for (int64_t i = 0; i < N; ++i) {
    const double px = pts[2 * i], py = pts[2 * i + 1];
    Poly P;
    const double B = 0.49 * std::min(Lx, Ly);
    P.n = 4;
    P.x[0] = -B; P.y[0] = -B; P.x[1] = B; P.y[1] = -B; P.x[2] = B; P.y[2] = B; P.x[3] = -B; P.y[3] = B;
    for (int k = 0; k < 4; ++k) P.nbr[k] = -1;
    int64_t ix, iy; cell_of(i, ix, iy);
    for (int64_t r = 0; r <= Rmax; ++r) {
      // stop once every point of ring r is farther than twice the largest vertex radius
      double R2 = 0.0;
      for (int k = 0; k < P.n; ++k) R2 = std::max(R2, P.x[k] * P.x[k] + P.y[k] * P.y[k]);
      double dmin = (double)(r - 1) * g;
      if (r >= 1 && dmin > 0.0 && dmin * dmin > 4.0 * R2) break;
      // a ring wider than the grid would revisit cells through the periodic wrap: cap per axis
      int64_t x0 = -r, x1 = r, y0 = -r, y1 = r;
      bool fullx = (2 * r + 1 >= Gx), fully = (2 * r + 1 >= Gy);
      for (int64_t dy = y0; dy <= y1; ++dy) {
        for (int64_t dx = x0; dx <= x1; ++dx) {
          if (std::max(std::llabs(dx), std::llabs(dy)) != r) continue;  // ring only
          // skip offsets that alias an already-visited grid cell through the wrap
          if (fullx && (dx < -(Gx / 2) || dx > (Gx - 1) / 2)) continue;
          if (fully && (dy < -(Gy / 2) || dy > (Gy - 1) / 2)) continue;
          int64_t cx = ((ix + dx) % Gx + Gx) % Gx, cy = ((iy + dy) % Gy + Gy) % Gy;
          for (int64_t t = start[cy * Gx + cx]; t < start[cy * Gx + cx + 1]; ++t) {
            int32_t j = items[t];
            if (j == i) continue;
            double ddx = min_image(pts[2 * j] - px, Lx), ddy = min_image(pts[2 * j + 1] - py, Ly);
            if (!clip(P, ddx, ddy, j)) return TILING_ECLIP;
          }
        }
      }
    }
    int n = P.n;
    for (int k = 0; k < n; ++k) if (P.nbr[k] < 0) return TILING_EOPEN;
    if (n > S) { info[0] = n; return TILING_ESTRIDE; }
    maxn = std::max<int64_t>(maxn, n);
    // canonical row start: vertex whose outgoing edge borders the smallest neighbour index
    int k0 = 0;
    for (int k = 1; k < n; ++k) if (P.nbr[k] < P.nbr[k0]) k0 = k;
    cvn[i] = n;
    for (int t = 0; t < n; ++t) cnbr[(size_t)i * S + t] = P.nbr[(k0 + t) % n];
    for (int t = 0; t < n; ++t) {
      int32_t b = cnbr[(size_t)i * S + t];                 // outgoing edge label
      int32_t a = cnbr[(size_t)i * S + (t + n - 1) % n];   // incoming edge label
      // counter-clockwise around the vertex the cells are (i, a, b)
      int32_t m = std::min((int32_t)i, std::min(a, b));
      int32_t vid = -1;
      if (m == (int32_t)i) {
        vid = (int32_t)V++;
        seen.push_back(1);
        // circumcentre of the three generators in the frame of the smallest index (= i)
        double ax = min_image(pts[2 * a] - px, Lx), ay = min_image(pts[2 * a + 1] - py, Ly);
        double bx = min_image(pts[2 * b] - px, Lx), by = min_image(pts[2 * b + 1] - py, Ly);
        // order the other two by index so that every cell would compute identical bits
        if (a > b) { std::swap(ax, bx); std::swap(ay, by); }
        double d = 2.0 * (ax * by - ay * bx);
        double a2 = ax * ax + ay * ay, b2 = bx * bx + by * by;
        double ux = (by * a2 - ay * b2) / d, uy = (ax * b2 - bx * a2) / d;
        if ((size_t)(2 * vid + 1) >= (size_t)(4 * N)) return TILING_ECOUNT;
        pos_xy[2 * vid] = wrap(px + ux, Lx);
        pos_xy[2 * vid + 1] = wrap(py + uy, Ly);
      } else {
        // look the vertex up in the row of the smallest-index cell m; seen from m the cyclic
        // order (m, next, nextnext) fixes its incoming/outgoing labels
        int32_t in_l, out_l;
        if (m == a) { in_l = b; out_l = (int32_t)i; } else { in_l = (int32_t)i; out_l = a; }
        int nm = cvn[m];
        const int32_t* rl = &cnbr[(size_t)m * S];
        for (int k = 0; k < nm; ++k)
          if (rl[k] == out_l && rl[(k + nm - 1) % nm] == in_l) { vid = cv[(size_t)m * S + k]; break; }
        if (vid < 0) return TILING_EMISMATCH;
        if (++seen[vid] > 3) return TILING_EMISMATCH;
      }
      cv[(size_t)i * S + t] = vid;
    }
  }
  info[0] = maxn; info[1] = V;
  if (V != 2 * N) return TILING_ECOUNT;
  for (int64_t v = 0; v < V; ++v) if (seen[v] != 3) return TILING_EMISMATCH;
  return tiling_from_rows(N, V, S, cvn, cv, vn, vc);
}

}  // extern "C"
