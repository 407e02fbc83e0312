// avm_step.cu — the per-timestep kernels of the AVM hot path for sm_100a.
//
// Paper order of one step (PAPER.md:62-64 §II.B, :104-108 §II.D; R6):
//   geometry -> forces -> move vertices -> rotate directors -> T1 test/update.
// Kernel schedule used here:
//   force_move   (thread/vertex)  rows a2+a3: F_v from the 3 incident cells' cached (a,p) records
//                                  and the 3 neighbour positions, Euler step of Eq. 4, wrap.
//   cell_update  (thread/cell)    rows a4+a1+a5: director noise, then area/perimeter of the MOVED
//                                  tiling (= the geometry the next step's forces need) and, from
//                                  the same edge vectors, detection of edges shorter than l_c.
//   t1_mark / t1_flip / t1_reset  rows a5-a7: eligibility, conflict rule, flip + list rewrite.
// Geometry is thus evaluated once per step on the positions the forces of the following step
// act on; after a flip the records of its four cells are refreshed in place, so every force is
// computed from the geometry of the current topology exactly as in the paper's cycle.
#include "avm_internal.cuh"

namespace avm {

static constexpr int kVertexBlock = 256;
static constexpr int kCellBlock = 128;
static constexpr int kT1Block = 128;
static constexpr int kT1Grid = 148 * 4;

// ---------------------------------------------------------------------------------------------
// rows a2 + a3: vertex forces (Eq. A2-A5) and displacement (Eq. 4, :56).
// Slot convention (R12): in cell c_k = vc[v][k] the CCW neighbours of v are next = vn[v][k],
// prev = vn[v][k+1], so no row search is needed.  With r_k = mi(h_{n_k} - h_v):
//   dA_{c_k}/dh_v = 1/2 (r_k.y - r_{k+1}.y, r_{k+1}.x - r_k.x)        (A4, R3)
//   dP_{c_k}/dh_v = -(rhat_k + rhat_{k+1})                             (A5, R2)
//   F_v = -sum_k [ a_k dA + p_k dP ],  a = 2K_A(A-A0), p = 2K_P(P-P0)  (A2, A3)
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double2 vertex_force(const double2 h, const double2 q0, const double2 q1,
                                                const double2 q2, const CellRec c0, const CellRec c1,
                                                const CellRec c2, const Consts& k) {
  const double r0x = min_image(q0.x - h.x, k.Lx, k.hLx), r0y = min_image(q0.y - h.y, k.Ly, k.hLy);
  const double r1x = min_image(q1.x - h.x, k.Lx, k.hLx), r1y = min_image(q1.y - h.y, k.Ly, k.hLy);
  const double r2x = min_image(q2.x - h.x, k.Lx, k.hLx), r2y = min_image(q2.y - h.y, k.Ly, k.hLy);
  const double s0 = r0x * r0x + r0y * r0y, s1 = r1x * r1x + r1y * r1y, s2 = r2x * r2x + r2y * r2y;
  const double i0 = s0 > 0.0 ? rsqrt(s0) : 0.0;   // zero-length edge contributes 0 (R15)
  const double i1 = s1 > 0.0 ? rsqrt(s1) : 0.0;
  const double i2 = s2 > 0.0 ? rsqrt(s2) : 0.0;
  const double u0x = r0x * i0, u0y = r0y * i0, u1x = r1x * i1, u1y = r1y * i1, u2x = r2x * i2, u2y = r2y * i2;
  // cell k uses (next, prev) = (r_k, r_{k+1})
  double fx = -0.5 * (c0.a * (r0y - r1y) + c1.a * (r1y - r2y) + c2.a * (r2y - r0y));
  double fy = -0.5 * (c0.a * (r1x - r0x) + c1.a * (r2x - r1x) + c2.a * (r0x - r2x));
  fx += c0.p * (u0x + u1x) + c1.p * (u1x + u2x) + c2.p * (u2x + u0x);
  fy += c0.p * (u0y + u1y) + c1.p * (u1y + u2y) + c2.p * (u2y + u0y);
  return make_double2(fx, fy);
}

__global__ void __launch_bounds__(kVertexBlock)
force_move_kernel(const Dev d, const Consts k) {
  const int v = blockIdx.x * kVertexBlock + threadIdx.x;
  if (v == 0) { d.ctr->n_short = 0; d.ctr->n_cand = 0; }   // T1 lists of the previous step are done
  if (v >= k.V) return;
  const double2 h = d.pos[v];
  const int n0 = d.vn[3 * v], n1 = d.vn[3 * v + 1], n2 = d.vn[3 * v + 2];
  const int e0 = d.vc[3 * v], e1 = d.vc[3 * v + 1], e2 = d.vc[3 * v + 2];
  const double2 q0 = d.pos[n0], q1 = d.pos[n1], q2 = d.pos[n2];
  const CellRec c0 = d.rec[e0], c1 = d.rec[e1], c2 = d.rec[e2];
  const double2 f = vertex_force(h, q0, q1, q2, c0, c1, c2, k);
  // Eq. 4: dh/dt = mu F + (v0/3) sum of the three unit directors (R5), directors of the start
  // of the step (R7); explicit Euler; wrap into the box (R13)
  const double vx = k.mu * f.x + k.v0_3 * (c0.nx + c1.nx + c2.nx);
  const double vy = k.mu * f.y + k.v0_3 * (c0.ny + c1.ny + c2.ny);
  const double x = wrap_box(h.x + k.dt * vx, k.Lx), y = wrap_box(h.y + k.dt * vy, k.Ly);
  if (!(isfinite(x) && isfinite(y))) atomicOr((unsigned long long*)&d.ctr->error, 1ull);
  d.pos_next[v] = make_double2(x, y);
}

// ---------------------------------------------------------------------------------------------
// rows a4 + a1 + a5: director update (R8, R16), geometry of the moved tiling
// (R14) and short-edge detection (R9).
// `pos` is the position buffer AFTER the move.  kUpdateTheta = false gives the plain geometry
// refresh used at creation / after avm_set_positions.
// ---------------------------------------------------------------------------------------------
template <bool kUpdateTheta, bool kDetect>
__global__ void __launch_bounds__(kCellBlock)
cell_update_kernel(const Dev d, const double2* __restrict__ pos, const Consts k, const unsigned long long step) {
  const int c = blockIdx.x * kCellBlock + threadIdx.x;
  if (c >= k.N) return;
  const int n = d.cvn[c];
  double th = d.theta[c];
  if (kUpdateTheta) {
    th += k.amp * director_noise(k.seed, step, (unsigned long long)(unsigned int)d.ctag[c]);
    d.theta[c] = th;
  }
  double sn, cs;
  sincos(th, &sn, &cs);

  const int4* row4 = reinterpret_cast<const int4*>(d.cv + (size_t)c * k.S);
  double acc = 0.0, per = 0.0;
  double rxp = 0.0, ryp = 0.0;
  int4 q = row4[0];
  const int first = q.x;
  int vprev = first;
  const double2 h0 = pos[first];
  for (int j = 1; j <= n; ++j) {
    if ((j & 3) == 0 && j < n) q = row4[j >> 2];
    const int sel = j & 3;
    int vj = sel == 0 ? q.x : sel == 1 ? q.y : sel == 2 ? q.z : q.w;
    double rx = 0.0, ry = 0.0;
    if (j < n) {
      const double2 hj = pos[vj];
      rx = min_image(hj.x - h0.x, k.Lx, k.hLx);
      ry = min_image(hj.y - h0.y, k.Ly, k.hLy);
    } else {
      vj = first;
    }
    acc += rxp * ry - ryp * rx;
    const double dx = rx - rxp, dy = ry - ryp;
    const double l2 = dx * dx + dy * dy;
    per += sqrt(l2);
    if (kDetect) {
      // each edge is seen by its two cells in opposite directions: report it from the cell that
      // traverses it from the smaller to the larger (current) vertex index
      if (l2 < k.lc2 && vprev < vj) {
        const unsigned int slot = atomicAdd(&d.ctr->n_short, 1u);
        d.short_list[slot] = make_int2(vprev, vj);
      }
    }
    rxp = rx; ryp = ry; vprev = vj;
  }
  CellRec r;
  r.a = k.KA2 * (0.5 * acc - k.A0);
  r.p = k.KP2 * (per - k.P0);
  r.nx = cs; r.ny = sn;
  d.rec[c] = r;
}

// Detection alone (test hooks avm_t1_pass / avm_debug_t1): thread per vertex, edge owned by the
// smaller current index.
__global__ void detect_short_edges_kernel(const Dev d, const Consts k) {
  const int v = blockIdx.x * blockDim.x + threadIdx.x;
  if (v >= k.V) return;
  const double2 h = d.pos[v];
  for (int s = 0; s < 3; ++s) {
    const int w = d.vn[3 * v + s];
    if (v < w) {
      const double2 q = d.pos[w];
      const double dx = min_image(q.x - h.x, k.Lx, k.hLx), dy = min_image(q.y - h.y, k.Ly, k.hLy);
      if (dx * dx + dy * dy < k.lc2) {
        const unsigned int slot = atomicAdd(&d.ctr->n_short, 1u);
        d.short_list[slot] = make_int2(v, w);
      }
    }
  }
}

__global__ void zero_counts_kernel(const Dev d) { d.ctr->n_short = 0; d.ctr->n_cand = 0; d.ctr->n_win = 0; }

// ---------------------------------------------------------------------------------------------
// rows a5 (eligibility) + a6 (conflict rule): R10, R11.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kT1Block)
t1_mark_kernel(const Dev d, const Consts k, const bool count_stats) {
  const unsigned int n_short = d.ctr->n_short;
  if (count_stats && blockIdx.x == 0 && threadIdx.x == 0) d.ctr->t1_short += n_short;
  for (unsigned int i = blockIdx.x * kT1Block + threadIdx.x; i < n_short; i += gridDim.x * kT1Block) {
    const int2 e = d.short_list[i];
    int v1 = e.x, v2 = e.y;
    unsigned int t1 = (unsigned int)d.vtag[v1], t2 = (unsigned int)d.vtag[v2];
    if (t1 > t2) { int tv = v1; v1 = v2; v2 = tv; unsigned int tt = t1; t1 = t2; t2 = tt; }
    int k1 = 0, k2 = 0;
#pragma unroll
    for (int s = 0; s < 3; ++s) {
      if (d.vn[3 * v1 + s] == v2) k1 = s;
      if (d.vn[3 * v2 + s] == v1) k2 = s;
    }
    // cyclic from the partner's slot the cells of u are (C0, C1, C2); C0 is left of u -> partner
    const int cL = d.vc[3 * v1 + k1], cE1 = d.vc[3 * v1 + (k1 + 1) % 3];
    const int cR = d.vc[3 * v2 + k2], cE2 = d.vc[3 * v2 + (k2 + 1) % 3];
    const bool distinct = cL != cR && cL != cE1 && cL != cE2 && cR != cE1 && cR != cE2 && cE1 != cE2;
    if (!distinct) continue;
    if (!(d.cvn[cL] > 3 && d.cvn[cR] > 3)) continue;             // no 2-gons (T2 absent)
    if (!(d.cvn[cE1] < k.S && d.cvn[cE2] < k.S)) {               // row would exceed the stride
      if (count_stats) {
        atomicAdd((unsigned long long*)&d.ctr->overflow_rejects, 1ull);
        atomicOr((unsigned long long*)&d.ctr->error, 2ull);
      }
      continue;
    }
    Cand cd;
    cd.v1 = v1; cd.v2 = v2; cd.k1 = k1; cd.k2 = k2;
    cd.cL = cL; cd.cR = cR; cd.cE1 = cE1; cd.cE2 = cE2;
    cd.key = ((unsigned long long)t1 << 32) | t2;
    cd.pad = 0;
    const unsigned int slot = atomicAdd(&d.ctr->n_cand, 1u);
    d.cand[slot] = cd;
    atomicMin(&d.minkey[cL], cd.key);
    atomicMin(&d.minkey[cR], cd.key);
    atomicMin(&d.minkey[cE1], cd.key);
    atomicMin(&d.minkey[cE2], cd.key);
  }
}

__device__ __forceinline__ void row_delete(int* __restrict__ row, int* __restrict__ cvn_c, int v) {
  const int n = *cvn_c;
  int j = 0;
  while (j < n && row[j] != v) ++j;
  for (int t = j; t + 1 < n; ++t) row[t] = row[t + 1];
  row[n - 1] = -1;
  *cvn_c = n - 1;
}
__device__ __forceinline__ void row_insert_after(int* __restrict__ row, int* __restrict__ cvn_c, int after, int v) {
  const int n = *cvn_c;
  int j = 0;
  while (j < n && row[j] != after) ++j;
  for (int t = n; t > j + 1; --t) row[t] = row[t - 1];
  row[j + 1] = v;
  *cvn_c = n + 1;
}

// ---------------------------------------------------------------------------------------------
// row a7: flip + rewrite (R9 geometry, R12 lists).  A candidate flips iff its key is the minimum
// recorded on all four of its cells (R11); winners therefore own disjoint cell quadruples and
// every word written below belongs to a vertex or row inside the winner's own quadruple.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kT1Block)
t1_flip_kernel(const Dev d, const Consts k) {
  const unsigned int n_cand = d.ctr->n_cand;
  unsigned int flips = 0, blocked = 0;
  for (unsigned int i = blockIdx.x * kT1Block + threadIdx.x; i < n_cand; i += gridDim.x * kT1Block) {
    const Cand c = d.cand[i];
    const bool win = d.minkey[c.cL] == c.key && d.minkey[c.cR] == c.key && d.minkey[c.cE1] == c.key &&
                     d.minkey[c.cE2] == c.key;
    if (!win) { ++blocked; continue; }
    ++flips;
    const int v1 = c.v1, v2 = c.v2, k1 = c.k1, k2 = c.k2;
    // geometry: rigid counter-clockwise quarter turn about the midpoint, new length 1.5 l_c (R9)
    const double2 h1 = d.pos[v1], h2 = d.pos[v2];
    const double dx = min_image(h2.x - h1.x, k.Lx, k.hLx), dy = min_image(h2.y - h1.y, k.Ly, k.hLy);
    const double l = sqrt(dx * dx + dy * dy);
    const double mx = h1.x + 0.5 * dx, my = h1.y + 0.5 * dy;
    double px = 0.0, py = 1.0;
    if (l > 0.0) { px = -dy / l; py = dx / l; }
    const double half = 0.75 * k.lc;
    d.pos[v2] = make_double2(wrap_box(mx + half * px, k.Lx), wrap_box(my + half * py, k.Ly));
    d.pos[v1] = make_double2(wrap_box(mx - half * px, k.Lx), wrap_box(my - half * py, k.Ly));
    // lists: u = ([w, x, y]; [C0, C1, C2]) cyclic from the partner slot
    //     -> ([w, y, z]; [C1, C2, C']), z = partner's old x, C' = partner's old C1 (R12)
    const int a1 = (k1 + 1) % 3, b1 = (k1 + 2) % 3, a2 = (k2 + 1) % 3, b2 = (k2 + 2) % 3;
    const int x1 = d.vn[3 * v1 + a1], y1 = d.vn[3 * v1 + b1];
    const int x2 = d.vn[3 * v2 + a2], y2 = d.vn[3 * v2 + b2];
    d.vn[3 * v1 + a1] = y1; d.vn[3 * v1 + b1] = x2;
    d.vc[3 * v1 + k1] = c.cE1; d.vc[3 * v1 + a1] = c.cR; d.vc[3 * v1 + b1] = c.cE2;
    d.vn[3 * v2 + a2] = y2; d.vn[3 * v2 + b2] = x1;
    d.vc[3 * v2 + k2] = c.cE2; d.vc[3 * v2 + a2] = c.cL; d.vc[3 * v2 + b2] = c.cE1;
#pragma unroll
    for (int s = 0; s < 3; ++s) {
      if (d.vn[3 * x1 + s] == v1) d.vn[3 * x1 + s] = v2;
    }
#pragma unroll
    for (int s = 0; s < 3; ++s) {
      if (d.vn[3 * x2 + s] == v2) d.vn[3 * x2 + s] = v1;
    }
    row_delete(d.cv + (size_t)c.cL * k.S, d.cvn + c.cL, v1);
    row_delete(d.cv + (size_t)c.cR * k.S, d.cvn + c.cR, v2);
    row_insert_after(d.cv + (size_t)c.cE1 * k.S, d.cvn + c.cE1, v1, v2);
    row_insert_after(d.cv + (size_t)c.cE2 * k.S, d.cvn + c.cE2, v2, v1);
    // refresh the cached geometry of the four cells (directors unchanged)
    const int cells[4] = {c.cL, c.cR, c.cE1, c.cE2};
#pragma unroll
    for (int t = 0; t < 4; ++t) {
      double A, P;
      cell_area_perimeter(d.pos, d.cv + (size_t)cells[t] * k.S, d.cvn[cells[t]], k, A, P);
      d.rec[cells[t]].a = k.KA2 * (A - k.A0);
      d.rec[cells[t]].p = k.KP2 * (P - k.P0);
    }
  }
  if (flips) atomicAdd((unsigned long long*)&d.ctr->t1_flips, (unsigned long long)flips);
  if (blocked) atomicAdd((unsigned long long*)&d.ctr->t1_blocked, (unsigned long long)blocked);
}

__global__ void __launch_bounds__(kT1Block)
t1_reset_kernel(const Dev d, const bool count_stats) {
  const unsigned int n_cand = d.ctr->n_cand;
  if (count_stats && blockIdx.x == 0 && threadIdx.x == 0) d.ctr->t1_candidates += n_cand;
  for (unsigned int i = blockIdx.x * kT1Block + threadIdx.x; i < n_cand; i += gridDim.x * kT1Block) {
    const Cand c = d.cand[i];
    d.minkey[c.cL] = ~0ull; d.minkey[c.cR] = ~0ull; d.minkey[c.cE1] = ~0ull; d.minkey[c.cE2] = ~0ull;
  }
}

// debug hook: winners without flipping; (tag_min, tag_max) pairs out
__global__ void t1_debug_kernel(const Dev d, int* cand_pairs, int* win_pairs, long long capacity) {
  const unsigned int n_cand = d.ctr->n_cand;
  for (unsigned int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_cand; i += gridDim.x * blockDim.x) {
    const Cand c = d.cand[i];
    if (cand_pairs && i < capacity) {
      cand_pairs[2 * i] = (int)(c.key >> 32);
      cand_pairs[2 * i + 1] = (int)(c.key & 0xffffffffu);
    }
    const bool win = d.minkey[c.cL] == c.key && d.minkey[c.cR] == c.key && d.minkey[c.cE1] == c.key &&
                     d.minkey[c.cE2] == c.key;
    if (win) {
      const unsigned int slot = atomicAdd(&d.ctr->n_win, 1u);
      if (win_pairs && slot < capacity) {
        win_pairs[2 * slot] = (int)(c.key >> 32);
        win_pairs[2 * slot + 1] = (int)(c.key & 0xffffffffu);
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// avm_compute_forces: unfused geometry and force kernels writing user-order outputs
// (App. A.1).  These do not touch the cached records, so they also serve as an
// in-library cross-check of the fused pass.
// ---------------------------------------------------------------------------------------------
__global__ void geometry_kernel(const Dev d, const Consts k, double2* __restrict__ ap, double* __restrict__ ap_user) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= k.N) return;
  double A, P;
  cell_area_perimeter(d.pos, d.cv + (size_t)c * k.S, d.cvn[c], k, A, P);
  ap[c] = make_double2(A, P);
  if (ap_user) {
    const int t = d.ctag[c];
    ap_user[2 * t] = A; ap_user[2 * t + 1] = P;
  }
}

__global__ void forces_kernel(const Dev d, const Consts k, const double2* __restrict__ ap, double* __restrict__ force_user) {
  const int v = blockIdx.x * blockDim.x + threadIdx.x;
  if (v >= k.V) return;
  const double2 h = d.pos[v];
  CellRec c[3];
  double2 q[3];
#pragma unroll
  for (int s = 0; s < 3; ++s) {
    q[s] = d.pos[d.vn[3 * v + s]];
    const double2 a = ap[d.vc[3 * v + s]];
    c[s].a = k.KA2 * (a.x - k.A0); c[s].p = k.KP2 * (a.y - k.P0); c[s].nx = 0.0; c[s].ny = 0.0;
  }
  const double2 f = vertex_force(h, q[0], q[1], q[2], c[0], c[1], c[2], k);
  const int t = d.vtag[v];
  force_user[2 * t] = f.x; force_user[2 * t + 1] = f.y;
}

// Energy, Eq. 1 / A1: block partial sums in a fixed order, finished by one
// block (deterministic, no floating-point atomics).
__global__ void energy_partial_kernel(const Dev d, const Consts k, double* __restrict__ partial) {
  __shared__ double sm[256];
  double e = 0.0;
  for (int c = blockIdx.x * 256 + threadIdx.x; c < k.N; c += gridDim.x * 256) {
    double A, P;
    cell_area_perimeter(d.pos, d.cv + (size_t)c * k.S, d.cvn[c], k, A, P);
    e += k.KA * (A - k.A0) * (A - k.A0) + k.KP * (P - k.P0) * (P - k.P0);
  }
  sm[threadIdx.x] = e;
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if (threadIdx.x < s) sm[threadIdx.x] += sm[threadIdx.x + s];
    __syncthreads();
  }
  if (threadIdx.x == 0) partial[blockIdx.x] = sm[0];
}
__global__ void energy_final_kernel(const Dev d, const double* __restrict__ partial, int n) {
  __shared__ double sm[256];
  double e = 0.0;
  for (int i = threadIdx.x; i < n; i += 256) e += partial[i];
  sm[threadIdx.x] = e;
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if (threadIdx.x < s) sm[threadIdx.x] += sm[threadIdx.x + s];
    __syncthreads();
  }
  if (threadIdx.x == 0) d.ctr->energy = sm[0];
}

__global__ void philox_words_kernel(unsigned long long seed, unsigned long long step, unsigned long long cell0,
                                    long long n, uint4* out) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = philox_for(seed, step, cell0 + (unsigned long long)i);
}

// ---------------------------------------------------------------------------------------------
// launchers
// ---------------------------------------------------------------------------------------------
static inline int cdiv(long long a, int b) { return (int)((a + b - 1) / b); }

// One timestep.  d.pos = positions at the start of the step, d.pos_next = buffer for the moved
// positions (the caller swaps them afterwards).
// ev (optional, 6 events): recorded before/after each kernel by avm_step_profile.
int launch_step(const Dev& d, const Consts& k, unsigned long long step, cudaStream_t s, cudaEvent_t* ev) {
  if (ev) cudaEventRecord(ev[0], s);
  force_move_kernel<<<cdiv(k.V, kVertexBlock), kVertexBlock, 0, s>>>(d, k);
  if (ev) cudaEventRecord(ev[1], s);
  Dev m = d;                      // from here on the moved positions are "the" positions
  m.pos = d.pos_next; m.pos_next = d.pos;
  cell_update_kernel<true, true><<<cdiv(k.N, kCellBlock), kCellBlock, 0, s>>>(m, m.pos, k, step);
  if (ev) cudaEventRecord(ev[2], s);
  t1_mark_kernel<<<kT1Grid, kT1Block, 0, s>>>(m, k, true);
  if (ev) cudaEventRecord(ev[3], s);
  t1_flip_kernel<<<kT1Grid, kT1Block, 0, s>>>(m, k);
  if (ev) cudaEventRecord(ev[4], s);
  t1_reset_kernel<<<kT1Grid, kT1Block, 0, s>>>(m, true);
  if (ev) cudaEventRecord(ev[5], s);
  return 5;
}

int launch_refresh_cells(const Dev& d, const Consts& k, cudaStream_t s) {
  cell_update_kernel<false, false><<<cdiv(k.N, kCellBlock), kCellBlock, 0, s>>>(d, d.pos, k, 0ull);
  return 1;
}

int launch_t1_pass_only(const Dev& d, const Consts& k, cudaStream_t s) {
  zero_counts_kernel<<<1, 1, 0, s>>>(d);
  detect_short_edges_kernel<<<cdiv(k.V, 256), 256, 0, s>>>(d, k);
  t1_mark_kernel<<<kT1Grid, kT1Block, 0, s>>>(d, k, true);
  t1_flip_kernel<<<kT1Grid, kT1Block, 0, s>>>(d, k);
  t1_reset_kernel<<<kT1Grid, kT1Block, 0, s>>>(d, true);
  zero_counts_kernel<<<1, 1, 0, s>>>(d);
  return 6;
}

int launch_t1_debug(const Dev& d, const Consts& k, int* cand_pairs, int* win_pairs, long long capacity, cudaStream_t s) {
  zero_counts_kernel<<<1, 1, 0, s>>>(d);
  detect_short_edges_kernel<<<cdiv(k.V, 256), 256, 0, s>>>(d, k);
  t1_mark_kernel<<<kT1Grid, kT1Block, 0, s>>>(d, k, false);
  t1_debug_kernel<<<kT1Grid, kT1Block, 0, s>>>(d, cand_pairs, win_pairs, capacity);
  t1_reset_kernel<<<kT1Grid, kT1Block, 0, s>>>(d, false);
  return 5;
}

int launch_compute_forces(const Dev& d, const Consts& k, double2* ap_scratch, double* force_user, double* ap_user, cudaStream_t s) {
  int n = 1;
  geometry_kernel<<<cdiv(k.N, 128), 128, 0, s>>>(d, k, ap_scratch, ap_user);
  if (force_user) { forces_kernel<<<cdiv(k.V, 256), 256, 0, s>>>(d, k, ap_scratch, force_user); ++n; }
  return n;
}

int launch_energy(const Dev& d, const Consts& k, double* partial, cudaStream_t s) {
  const int nb = 148 * 2;
  energy_partial_kernel<<<nb, 256, 0, s>>>(d, k, partial);
  energy_final_kernel<<<1, 256, 0, s>>>(d, partial, nb);
  return 2;
}

int launch_philox_words(unsigned long long seed, unsigned long long step, unsigned long long cell0, long long n,
                        uint32_t* out, cudaStream_t s) {
  if (n <= 0) return 0;
  philox_words_kernel<<<cdiv(n, 256), 256, 0, s>>>(seed, step, cell0, n, reinterpret_cast<uint4*>(out));
  return 1;
}

}  // namespace avm
