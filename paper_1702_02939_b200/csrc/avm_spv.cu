// avm_spv.cu — the GPU-only parts of one self-propelled-Voronoi (SPV) step on a FIXED triangulation
// (second half; section II.C, App. A.2 :171-200).
//
// The triangulation is the dual reading of the three topology lists the simulation already holds
// (PAPER.md:66): vertex v <-> Delaunay triangle with corners vc[v][0..2]; row c of cellVertices = the
// triangles (Voronoi vertices) around cell c, counter-clockwise; vn[v][k] = the adjacent triangles.
// The cell positions r_i are a caller-owned array in USER order.  Stages (paper order):
//   spv_voronoi       PAPER.md:82-84   Voronoi vertex of every triangle = circumcentre of its three
//                                      cells, saved as the simulation's vertex positions; the cell
//                                      pass of the AVM path then gives every area and perimeter
//   spv_dedh          App. A.1         dE/dh_v of every Voronoi vertex (the vertex-model derivative)
//   spv_cell_force    PAPER.md:86-88   "force sets" f_(i,v) = -(dh_v/dr_i)^T dE/dh_v (Eq. A6-A7) and their
//                                      sum over the row of cell i, in row order
//   spv_move          Eq. 3, :54, :92  r_i += dt (mu F_i + v0 n_i), wrap; director noise
//   spv_test          PAPER.md:94      empty-circumcircle test of every triangle against the cell
//                                      opposite each of its edges; count and per-cell flags
// The CPU/CGAL repair of PAPER.md:96-100 is out of scope.  Readings S1-S3: DESIGN.md section 14.
//
// dh_v/dr_i (reading S1; Eq. A11-A14 are garbled in PAPER.md).  h is equidistant from its corners:
//   M h = q,  M = [ (r_j - r_i)^T ; (r_k - r_i)^T ],  q = 1/2 ( |r_j|^2 - |r_i|^2 , |r_k|^2 - |r_i|^2 ).
// Differentiating with respect to r_i gives M dh = (1, 1)^T (h - r_i) . dr_i, i.e. the rank-one matrix
//   dh/dr_i = w (h - r_i)^T,   w = M^-1 (1, 1)^T = ( c_y - b_y , b_x - c_x ) / (b_x c_y - b_y c_x),
// with b = r_j - r_i, c = r_k - r_i, so that f_(i,v) = -(w . g_v) (h_v - r_i), g_v = dE/dh_v.
#include "avm_internal.cuh"

namespace avm {

struct Circle { double2 r0, u; double R2; };   // corner 0, centre relative to it, squared radius

__device__ __forceinline__ double2 cell_xy_ld(const double* __restrict__ cell_xy, int tag) {
  return make_double2(cell_xy[2 * tag], cell_xy[2 * tag + 1]);
}

// circumcircle of triangle v from the current cell positions (minimum image relative to corner 0)
__device__ __forceinline__ Circle circumcircle(const Dev& d, const Consts& k, const double* __restrict__ cell_xy, int v) {
  const int c0 = d.vc[v], c1 = d.vc[k.Vs + v], c2 = d.vc[2 * k.Vs + v];
  Circle o;
  o.r0 = cell_xy_ld(cell_xy, d.ctag[c0]);
  const double2 r1 = cell_xy_ld(cell_xy, d.ctag[c1]), r2 = cell_xy_ld(cell_xy, d.ctag[c2]);
  const double bx = min_image(r1.x - o.r0.x, k.Lx, k.hLx), by = min_image(r1.y - o.r0.y, k.Ly, k.hLy);
  const double cx = min_image(r2.x - o.r0.x, k.Lx, k.hLx), cy = min_image(r2.y - o.r0.y, k.Ly, k.hLy);
  const double D = 2.0 * (bx * cy - by * cx);
  const double b2 = bx * bx + by * by, c2n = cx * cx + cy * cy;
  o.u = make_double2((cy * b2 - by * c2n) / D, (bx * c2n - cx * b2) / D);
  o.R2 = o.u.x * o.u.x + o.u.y * o.u.y;
  return o;
}

// Voronoi vertices, saved as the simulation's vertex positions (internal order) and,
// optionally, in user order
__global__ void spv_voronoi_kernel(const Dev d, const Consts k, const double* __restrict__ cell_xy, double* __restrict__ voronoi_user) {
  const int v = blockIdx.x * blockDim.x + threadIdx.x;
  if (v >= k.V) return;
  const Circle o = circumcircle(d, k, cell_xy, v);
  double2 h = make_double2(wrap_box(o.r0.x + o.u.x, k.Lx), wrap_box(o.r0.y + o.u.y, k.Ly));
  if (!(isfinite(h.x) && isfinite(h.y))) { atomicOr((unsigned long long*)&d.ctr->error, 1ull); h = o.r0; }   // degenerate triangle
  pos_st(d.pos + v, h, k);
  const int t = d.vtag[v];
  // as avm_set_positions: the positions were replaced, not moved, so the unwrapped positions and the reference of the
  // mean-square displacement restart from them (stale image counts would pair with unrelated positions)
  d.msd_ref[t] = pos_ld(d.pos + v, k);
  d.img[t] = make_int2(0, 0);
  if (voronoi_user) { voronoi_user[2 * t] = h.x; voronoi_user[2 * t + 1] = h.y; }
}

// App. A.1: g_v = dE/dh_v = -(vertex force) from the cached (2 K_A (A - A0), 2 K_P (P - P0)) of the three cells
__global__ void spv_dedh_kernel(const Dev d, const Consts k, double2* __restrict__ g) {
  const int v = blockIdx.x * blockDim.x + threadIdx.x;
  if (v >= k.V) return;
  const double2 h = pos_ld(d.pos + v, k);
  double2 q[3];
  CellRec c[3];
#pragma unroll
  for (int s = 0; s < 3; ++s) {
    q[s] = pos_ld(d.pos + d.vn[s * k.Vs + v], k);
    c[s] = rec_ld_plain(d.rec + d.vc[s * k.Vs + v]);
  }
  const double2 f = vertex_force(h, q[0], q[1], q[2], c[0], c[1], c[2], k);
  g[v] = make_double2(-f.x, -f.y);
}

// PAPER.md:86-88, Eq. A6-A7: force sets of cell c and their sum in row order.  force_int: internal order
// (read by the move); force_user, sets_user ([N][S][2]): optional outputs in user order.
__global__ void spv_cell_force_kernel(const Dev d, const Consts k, const double* __restrict__ cell_xy, const double2* __restrict__ g,
                                      double2* __restrict__ force_int, double* __restrict__ force_user, double* __restrict__ sets_user) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= k.N) return;
  const int t = d.ctag[c], n = d.cvn[c];
  const double2 ri = cell_xy_ld(cell_xy, t);
  double Fx = 0.0, Fy = 0.0;
  for (int j = 0; j < k.S; ++j) {
    double fx = 0.0, fy = 0.0;
    if (j < n) {
      const int v = row_entry(d.cv, k.N, c, j);
      const int c0 = d.vc[v], c1 = d.vc[k.Vs + v], c2 = d.vc[2 * k.Vs + v];
      // the other two corners, cyclically after this cell
      const int cj = c0 == c ? c1 : c1 == c ? c2 : c0, ck = c0 == c ? c2 : c1 == c ? c0 : c1;
      const double2 rj = cell_xy_ld(cell_xy, d.ctag[cj]), rk = cell_xy_ld(cell_xy, d.ctag[ck]);
      const double bx = min_image(rj.x - ri.x, k.Lx, k.hLx), by = min_image(rj.y - ri.y, k.Ly, k.hLy);
      const double cx = min_image(rk.x - ri.x, k.Lx, k.hLx), cy = min_image(rk.y - ri.y, k.Ly, k.hLy);
      const double det = bx * cy - by * cx;
      const double wx = (cy - by) / det, wy = (bx - cx) / det;
      const double2 h = pos_ld(d.pos + v, k);
      const double hx = min_image(h.x - ri.x, k.Lx, k.hLx), hy = min_image(h.y - ri.y, k.Ly, k.hLy);
      const double2 gv = g[v];
      const double coef = -(wx * gv.x + wy * gv.y);
      fx = coef * hx; fy = coef * hy;
      Fx += fx; Fy += fy;
    }
    if (sets_user) {
      sets_user[((size_t)t * k.S + j) * 2] = fx;
      sets_user[((size_t)t * k.S + j) * 2 + 1] = fy;
    }
  }
  force_int[c] = make_double2(Fx, Fy);
  if (force_user) { force_user[2 * t] = Fx; force_user[2 * t + 1] = Fy; }
}

// Eq. 3: explicit Euler with the director of the start of the step, wrap; then the director
// noise of PAPER.md:50 (R8, R16: the same Philox-keyed update as the AVM path)
__global__ void spv_move_kernel(const Dev d, const Consts k, double* __restrict__ cell_xy, const double2* __restrict__ force_int,
                                const double v0, const unsigned long long step) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= k.N) return;
  const int t = d.ctag[c];
  double th = d.theta[c];
  double sn, cs;
  sincos_any(th, &sn, &cs);
  const double2 F = force_int[c];
  double x = cell_xy[2 * t] + k.dt * (k.mu * F.x + v0 * cs);
  double y = cell_xy[2 * t + 1] + k.dt * (k.mu * F.y + v0 * sn);
  x = wrap_box(x, k.Lx); y = wrap_box(y, k.Ly);
  if (!(isfinite(x) && isfinite(y))) atomicOr((unsigned long long*)&d.ctr->error, 1ull);
  cell_xy[2 * t] = x; cell_xy[2 * t + 1] = y;
  th += k.amp * director_noise(k, step, (unsigned long long)(unsigned int)t);
  d.theta[c] = th;
}

// one thread per triangle tests its circumcircle against the cell opposite each of its three
// edges (reading S2), strictly (S3).  counts[0] += failed tests; flags (user order, optional): the corners of a
// failing triangle and the intruding cell.
__global__ void spv_test_kernel(const Dev d, const Consts k, const double* __restrict__ cell_xy, unsigned long long* __restrict__ counts,
                                int* __restrict__ flags, const unsigned long long step_rel) {
  const int v = blockIdx.x * blockDim.x + threadIdx.x;
  if (v >= k.V) return;
  const Circle o = circumcircle(d, k, cell_xy, v);
  const int c0 = d.vc[v], c1 = d.vc[k.Vs + v], c2 = d.vc[2 * k.Vs + v];
  int nfail = 0;
  for (int e = 0; e < 3; ++e) {
    const int w = d.vn[e * k.Vs + v];
    int opp = -1;
    for (int m = 0; m < 3; ++m) {
      const int cand = d.vc[m * k.Vs + w];
      if (cand != c0 && cand != c1 && cand != c2) opp = cand;
    }
    if (opp < 0) continue;                       // degenerate neighbourhood (the two triangles share all corners)
    const double2 ro = cell_xy_ld(cell_xy, d.ctag[opp]);
    const double dx = min_image(ro.x - o.r0.x, k.Lx, k.hLx) - o.u.x, dy = min_image(ro.y - o.r0.y, k.Ly, k.hLy) - o.u.y;
    if (dx * dx + dy * dy < o.R2) {
      ++nfail;
      if (flags) { flags[d.ctag[opp]] = 1; flags[d.ctag[c0]] = 1; flags[d.ctag[c1]] = 1; flags[d.ctag[c2]] = 1; }
    }
  }
  if (nfail) {
    atomicAdd(counts, (unsigned long long)nfail);
    atomicMin(counts + 1, step_rel);              // first step of the call after which the triangulation was invalid
  }
}

static inline int cdiv_spv(long long a, int b) { return (int)((a + b - 1) / b); }

int launch_spv_voronoi(const Dev& d, const Consts& k, const double* cell_xy, double* voronoi_user, cudaStream_t s) {
  spv_voronoi_kernel<<<cdiv_spv(k.V, 256), 256, 0, s>>>(d, k, cell_xy, voronoi_user);
  return 1;
}
int launch_spv_forces(const Dev& d, const Consts& k, const double* cell_xy, double2* g_scratch, double2* force_int, double* force_user,
                      double* sets_user, cudaStream_t s) {
  spv_dedh_kernel<<<cdiv_spv(k.V, 256), 256, 0, s>>>(d, k, g_scratch);
  spv_cell_force_kernel<<<cdiv_spv(k.N, 128), 128, 0, s>>>(d, k, cell_xy, g_scratch, force_int, force_user, sets_user);
  return 2;
}
int launch_spv_move(const Dev& d, const Consts& k, double* cell_xy, const double2* force_int, double v0, unsigned long long step,
                    cudaStream_t s) {
  spv_move_kernel<<<cdiv_spv(k.N, 256), 256, 0, s>>>(d, k, cell_xy, force_int, v0, step);
  return 1;
}
int launch_spv_test(const Dev& d, const Consts& k, const double* cell_xy, unsigned long long* counts, int* flags,
                    unsigned long long step_rel, cudaStream_t s) {
  spv_test_kernel<<<cdiv_spv(k.V, 256), 256, 0, s>>>(d, k, cell_xy, counts, flags, step_rel);
  return 1;
}

}  // namespace avm
