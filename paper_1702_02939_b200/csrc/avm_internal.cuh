// avm_internal.cuh — shared declarations of the CUDA path (sm_100a).  Not part of the C ABI.
//
// Notation follows the paper (PAPER.md = /root/reference/PAPER.md): h = vertex position,
// A/P = cell area / perimeter, theta = director angle, cellVertices / vertexNeighbors /
// vertexCellNeighbors = the three flat topology lists of PAPER.md:66.  R-numbers = DESIGN.md.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/avm.h"
#include "avm_math.cuh"

namespace avm {

// Per-cell record gathered by the force/move kernel: one 32-byte sector per cell.
//   a  = 2 K_A (A_c - A0)   (Eq. A3 prefactor)
//   p  = 2 K_P (P_c - P0)
//   nx = cos(theta_c), ny = sin(theta_c)   (director)
struct __align__(32) CellRec { double a, p, nx, ny; };

// ---------------------------------------------------------------------------------------------
// Storage formats.  Default build: positions double2, records 4 doubles (everything fp64).
// -DAVM_MIXED=1 (libavm_b200_mixed.so; PAPER.md:120 shows a single-precision variant):
// reduced-precision STORAGE, fp64 arithmetic.  Positions live on a fixed-point grid of 2^-32 box lengths
// per axis (8 bytes instead of 16; the periodic box is the natural range of the integer), records are
// four floats (16 bytes instead of 32).  Every kernel unpacks to double on load and packs on store,
// so the arithmetic of the step is the same code in both builds; the accuracy contract is in avm.h.
// ---------------------------------------------------------------------------------------------
#ifndef AVM_MIXED
#define AVM_MIXED 0
#endif
#if AVM_MIXED
typedef uint2 pos_t;
struct __align__(16) rec_t { float a, p, nx, ny; };
#else
typedef double2 pos_t;
typedef CellRec rec_t;
#endif

// Per-cell parameters of Eq. 1 (NEXT-4): preferred area / perimeter and moduli.
struct __align__(32) CellPar { double A0, P0, KA, KP; };

// One eligible T1 candidate (R10), decoded once by the detecting thread and reused by the flip.
struct __align__(16) Cand {
  int v1, v2;           // v1 = endpoint with the smaller tag
  int k1, k2;           // slot of v2 in v1, slot of v1 in v2
  int cL, cR, cE1, cE2; // the two cells sharing the edge, the two end cells (R12)
  unsigned long long key;  // (tag(v1) << 32) | tag(v2)  (R11)
  int sx1, sx2;         // slot of v1 in x1, slot of v2 in x2
  int x1, y1, x2, y2;   // the other two neighbours of v1 (cyclic after v2) and of v2 (cyclic after v1)
};

struct Counters {
  // candidate list length, double-buffered by step parity: the list of step s is flipped by
  // t1_flip(s) and its per-cell minimum keys are cleared by the prologue of force_move(s+1)
  unsigned int n_cand[4];   // [0], [1]: the step's list by step parity; [2], [3]: lists of repeated passes (NEXT-1)
  unsigned int n_win;     // winners (debug hook); short edges at creation
  unsigned int feedback_sink;   // target of Dev::feedback when no mapped host word is available
  unsigned int fb_last;         // T1 load last written to Dev::feedback (it is rewritten only when the load crosses the schedule threshold)
  unsigned int pad0[25];
  // fused schedule, zeroed by the cell pass of every step.  Each on a 128-byte line of its own: the
  // first is hammered by claiming atomics while waiting warps poll the second.
  unsigned int next_cand; // next candidate index to be claimed
  unsigned int pad1[31];
  unsigned int flip_done; // candidates decided so far
  unsigned int pad2[31];
  unsigned int bar;       // arrival counter of the persistent kernel's grid barrier (zeroed by the host before each launch)
  unsigned int pad3[31];
  long long t1_short, t1_candidates, t1_flips, t1_blocked, overflow_rejects, error;
  double obs[16];  // observables of the latest avm_energy / avm_observe call (slots: avm_step.cu)
  unsigned long long spv[2];   // SPV circumcircle test (avm_spv.cu): failed tests of the latest step, first failing step of the call
};

// Up to this many T1 candidates a step leaves its flips to the next force/move launch (two launches per
// step); beyond, the stand-alone T1 kernel is faster.
#ifndef AVM_FUSED_MAX_CANDIDATES
#define AVM_FUSED_MAX_CANDIDATES 1024
#endif

// Model constants, passed by value to every kernel.
struct Consts {
  int N, V, S;
  int Vs;                    // plane stride of vn / vc (V rounded up to 64 entries)
  double Lx, Ly, hLx, hLy;
  double KA2, KP2, A0, P0;   // KA2 = 2 K_A, KP2 = 2 K_P
  double KA, KP;
  double v0_3, mu, dt;       // v0_3 = v0 / 3 (Eq. 4 with n = 3, R5)
  double amp;                // sqrt(2 Dr dt) (R8)
  double lc, lc2;
  double ux, uy, iux, iuy;   // mixed build: grid unit Lx / 2^32, Ly / 2^32 and their inverses
  int flag_dirty;            // 1: the marking thread flags the vertices of a candidate's cells (two-launch schedule only)
  int clear_dirty;           // 1: the cell pass clears the bitmap the force/move launch of this step swept with
  int nw;                    // words per dirty bitmap (V/32 rounded up to a multiple of 32)
  int fm_grid;               // CTAs of the persistent force/move grid (a whole number per SM, set at create)
  int per_cell;              // 1: A0_i, P0_i, K_A,i, K_P,i per cell (Dev::par, Eq. 1), 0: the uniform values of Eq. A1
  int cap_a;                 // capacity of the step's candidate list (3N: every edge of the tiling)
  unsigned long long seed;
  uint2 rkey[10];            // Philox round keys of `seed` (the key schedule is uniform: done once on the host)
};

// Pointers into the caller's workspace (current buffer set).
//
// Layout: everything is structure-of-arrays.
//   vn, vc : three planes of Vs ints each: vn[k*Vs + v] = k-th neighbour of v (slot convention R12)
//   cv     : fixed-stride padded rows stored as S/4 planes of int4: entries 4q..4q+3 of cell c are
//            cv[q*N + c]; unused entries repeat entry 0 (always a valid index).  A warp reads 32 consecutive cells' quads with one
//            fully coalesced 128-bit load per plane, and cells with <= 8 vertices (96 %) never
//            touch planes 2, 3.
struct Dev {
  pos_t* pos;         // [V] current positions
  pos_t* pos_next;    // [V] written by force_move, then swapped
  int* vn;            // [3*Vs] vertexNeighbors planes
  int* vc;            // [3*Vs] vertexCellNeighbors planes
  int4* cv;           // [(S/4)*N] cellVertices planes
  int* cvn;           // [N] cellVertexNum
  double* theta;      // [N]
  rec_t* rec;         // [N]
  int* vtag;          // [V] user index of each vertex
  int* ctag;          // [N] user index of each cell
  unsigned long long* minkey;  // [N] per-cell minimum candidate key, ~0 when idle
  Cand* cand;         // [3N]
  unsigned int* dirty; // [2][nw] bit v of buffer (s & 1): vertex v belongs to a cell of a T1 candidate found in
                       // step s.  Written only by the cell pass of step s, read only by the force/move launch
                       // of step s+1 (read-only for that whole launch), cleared by the cell pass of step s+1.
  CellPar* par;       // [N] (A0_i, P0_i, K_A,i, K_P,i), internal order; read only when Consts::per_cell (NEXT-4)
  int2* img;          // [V] USER order: how many box lengths each vertex has left through the boundary (NEXT-2, MSD)
  double2* msd_ref;   // [V] USER order: unwrapped positions at the reference time of the mean-square displacement
  unsigned long long* img_stamp; // [V] USER order: step + 1 of the latest image-count update made by a post-flip mover of the
                                 // two-launch schedule (those may move a vertex more than once per step; the count is applied once)
  unsigned int* estamp; // [3*Vs] per directed half-edge (slot plane, owner vertex): id of the repeated pass that tested it last
  Counters* ctr;
  unsigned int* feedback; // mapped HOST word: every force/move launch reports the candidate count of the previous step
                          // (read by the host without synchronising, to choose the schedule of later steps)
};

// ---------------------------------------------------------------------------------------------
// device helpers
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double min_image(double d, double L, double hL) {
  // positions stay in [0,L): one correction suffices (R13)
  if (d > hL) d -= L; else if (d < -hL) d += L;
  return d;
}
__device__ __forceinline__ double wrap_box(double x, double L) {
  if (x < 0.0) x += L;
  if (x >= L) x -= L;
  return x;
}
__device__ __forceinline__ unsigned int hi_word(double x) { return (unsigned int)__double2hiint(x); }

// ---- packing / unpacking of the storage formats (identity in the fp64 build) ----
#if AVM_MIXED
__device__ __forceinline__ double2 pos_unpack(const pos_t q, const Consts& k) {
  return make_double2(__dmul_rn((double)q.x, k.ux), __dmul_rn((double)q.y, k.uy));      // ux = Lx / 2^32
}
__device__ __forceinline__ pos_t pos_pack(const double2 h, const Consts& k) {
  // h in [0, L): nearest grid point; a coordinate that rounds up to the box length wraps to 0
  return make_uint2((unsigned int)__double2ull_rn(__dmul_rn(h.x, k.iux)), (unsigned int)__double2ull_rn(__dmul_rn(h.y, k.iuy)));
}
__device__ __forceinline__ CellRec rec_unpack(const float4 f) { CellRec r; r.a = f.x; r.p = f.y; r.nx = f.z; r.ny = f.w; return r; }
#else
__device__ __forceinline__ double2 pos_unpack(const pos_t q, const Consts&) { return q; }
__device__ __forceinline__ pos_t pos_pack(const double2 h, const Consts&) { return h; }
#endif
__device__ __forceinline__ double2 pos_ld(const pos_t* p, const Consts& k) { return pos_unpack(*p, k); }
__device__ __forceinline__ double2 pos_ldg(const pos_t* p, const Consts& k) { return pos_unpack(__ldg(p), k); }
__device__ __forceinline__ double2 pos_ldcg(const pos_t* p, const Consts& k) { return pos_unpack(__ldcg(p), k); }
__device__ __forceinline__ void pos_st(pos_t* p, const double2 h, const Consts& k) { *p = pos_pack(h, k); }
// the value a stored position reads back as (the packing is not the identity in the mixed build)
__device__ __forceinline__ double2 pos_round(const double2 h, const Consts& k) { return pos_unpack(pos_pack(h, k), k); }
#if AVM_MIXED
__device__ __forceinline__ CellRec rec_ld_plain(const rec_t* p) { return rec_unpack(*reinterpret_cast<const float4*>(p)); }
__device__ __forceinline__ CellRec rec_ldcg(const rec_t* p) { return rec_unpack(__ldcg(reinterpret_cast<const float4*>(p))); }
__device__ __forceinline__ void rec_st_ap(rec_t* p, double a, double pp) { *reinterpret_cast<float2*>(p) = make_float2((float)a, (float)pp); }
#else
__device__ __forceinline__ CellRec rec_ld_plain(const rec_t* p) { return *p; }
__device__ __forceinline__ CellRec rec_ldcg(const rec_t* p) {
  const double2* r = reinterpret_cast<const double2*>(p);
  const double2 ap = __ldcg(r), nn = __ldcg(r + 1);
  CellRec c; c.a = ap.x; c.p = ap.y; c.nx = nn.x; c.ny = nn.y;
  return c;
}
__device__ __forceinline__ void rec_st_ap(rec_t* p, double a, double pp) { p->a = a; p->p = pp; }
#endif

// entry j of cell c's row
__device__ __forceinline__ int& row_entry(int4* cv, int N, int c, int j) {
  return reinterpret_cast<int*>(cv + (size_t)(j >> 2) * N + c)[j & 3];
}
__device__ __forceinline__ int row_entry(const int4* cv, int N, int c, int j) {
  return reinterpret_cast<const int*>(cv + (size_t)(j >> 2) * N + c)[j & 3];
}

// parameters of cell c: Eq. 1 per cell or the uniform values of Eq. A1
__device__ __forceinline__ CellPar cell_params(const Dev& d, const Consts& k, int c) {
  if (k.per_cell) return d.par[c];
  CellPar q; q.A0 = k.A0; q.P0 = k.P0; q.KA = k.KA; q.KP = k.KP;
  return q;
}
// the cached record of a cell from its area and perimeter: a = 2 K_A (A - A0), p = 2 K_P (P - P0) (Eq. A3)
__device__ __forceinline__ void rec_from_geometry(const CellPar& q, double A, double P, double& a, double& p) {
  a = (2.0 * q.KA) * (A - q.A0);
  p = (2.0 * q.KP) * (P - q.P0);
}
// Image counts of a wrapped coordinate (NEXT-2): wrap_box with the number of box lengths added
__device__ __forceinline__ double wrap_box_count(double x, double L, int& n) {
  if (x < 0.0) { x += L; --n; }
  if (x >= L) { x -= L; ++n; }
  return x;
}

// Square roots of squared lengths.  Every squared length in this library is formed as
//   l2 = dx*dx + dy*dy + kTiny            (kTiny = 1e-300, far below one ulp of any real length)
// so that l2 is never zero or subnormal: a zero-length edge then yields rsqrt = 1e150 and
// r * rsqrt = 0 exactly, i.e. it contributes nothing (R15), without a compare/select per edge.
//
// MUFU.RSQ64H seed y0 (relative error ~2^-22) followed by one third-order correction, with
// e = 1 - x y0^2:   1/sqrt(x) = y0 (1 + e/2 + 3 e^2/8 + O(e^3)),   sqrt(x) = x y0 (1 + e/2 + 3 e^2/8 + ...)
// which leaves ~2^-66 before the final rounding.  5 FP64 operations each.
static constexpr double kTiny = 1e-300;
__device__ __forceinline__ double rsqrt_seed(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  return y;
}
__device__ __forceinline__ double rsqrt_pos(double x) {   // x >= kTiny
  const double y = rsqrt_seed(x);
  const double t = __dmul_rn(x, y);
  const double e = __fma_rn(-t, y, 1.0);
  const double p = __fma_rn(0.375, e, 0.5);
  return __fma_rn(__dmul_rn(y, e), p, y);
}
__device__ __forceinline__ double sqrt_pos(double x) {    // x >= kTiny
  const double y = rsqrt_seed(x);
  const double g = __dmul_rn(x, y);
  const double e = __fma_rn(-g, y, 1.0);
  const double p = __fma_rn(0.375, e, 0.5);
  return __fma_rn(__dmul_rn(g, e), p, g);
}

// Philox4x32-10 (Salmon et al., SC'11; R16).  Counter (c0..c3), key (k0,k1); round r uses the
// key (k0 + r 0x9E3779B9, k1 + r 0xBB67AE85).
__host__ __device__ __forceinline__ uint2 philox_round_key(unsigned long long seed, int r) {
  return make_uint2((unsigned)seed + (unsigned)r * 0x9E3779B9u, (unsigned)(seed >> 32) + (unsigned)r * 0xBB67AE85u);
}
__device__ __forceinline__ uint4 philox_round(uint4 c, uint2 k) {
  const unsigned int hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
  const unsigned int hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
  return make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
}
__device__ __forceinline__ uint4 philox_for(unsigned long long seed, unsigned long long step,
                                            unsigned long long cell) {
  uint4 c = make_uint4((unsigned)step, (unsigned)(step >> 32), (unsigned)cell, (unsigned)(cell >> 32));
#pragma unroll
  for (int r = 0; r < 10; ++r) c = philox_round(c, philox_round_key(seed, r));
  return c;
}
// the same block with the round keys taken from the kernel constants
__device__ __forceinline__ uint4 philox_for(const Consts& k, unsigned long long step, unsigned long long cell) {
  uint4 c = make_uint4((unsigned)step, (unsigned)(step >> 32), (unsigned)cell, (unsigned)(cell >> 32));
#pragma unroll
  for (int r = 0; r < 10; ++r) c = philox_round(c, k.rkey[r]);
  return c;
}
// Standard normal from one Philox block: two 52-bit uniforms in (0,1), Box-Muller cosine branch (R16).
// u = (m + 1/2) 2^-52 with m the top 52 bits of a 64-bit word.  Built without an integer->double
// conversion: the double with exponent 0 and mantissa m is 1 + m 2^-52, and adding (2^-53 - 1) is exact.
__device__ __forceinline__ double uniform52(unsigned int lo, unsigned int hi) {
  const double one_plus = __hiloint2double((int)(0x3ff00000u | (hi >> 12)), (int)((hi << 20) | (lo >> 12)));
  return __dadd_rn(one_plus, 1.1102230246251565e-16 - 1.0);
}
__device__ __forceinline__ double director_noise(const Consts& k, unsigned long long step, unsigned long long cell) {
  const uint4 x = philox_for(k, step, cell);
  const double u1 = uniform52(x.x, x.y), u2 = uniform52(x.z, x.w);
  return sqrt_pos(-2.0 * log_unit(u1)) * cos_2pi(u2);   // -2 ln u1 >= 2.2e-16 > kTiny
}

// One edge of the shoelace / perimeter sums (Eq. A1 inputs, R14): previous unwrapped vertex
// (rxp, ryp), current (rx, ry), both relative to the row's first vertex.  Explicit rounding
// intrinsics fix the operation order, so every kernel that sums a cell (the per-step pass, the T1
// refresh, avm_compute_forces) produces the same bits.  Returns the squared edge length.
__device__ __forceinline__ double geom_edge(double rxp, double ryp, double rx, double ry, double& acc, double& per) {
  acc = __fma_rn(rxp, ry, acc);
  acc = __fma_rn(-ryp, rx, acc);
  const double dx = __dsub_rn(rx, rxp), dy = __dsub_rn(ry, ryp);
  const double l2 = __fma_rn(dx, dx, __fma_rn(dy, dy, kTiny));
  per = __dadd_rn(per, sqrt_pos(l2));
  return l2;
}

// Area and perimeter of one cell from its row, one thread, plain loads (safe right after this
// warp rewrote the row).  Used by the cold paths: T1 refresh, avm_compute_forces, energy.
__device__ __forceinline__ void cell_area_perimeter(const pos_t* pos, const int4* cv, int c, int n,
                                                    const Consts& k, double& A, double& P) {
  const double2 h0 = pos_ld(pos + row_entry(cv, k.N, c, 0), k);
  double rxp = 0.0, ryp = 0.0, acc = 0.0, per = 0.0;
  for (int j = 1; j <= n; ++j) {
    double rx = 0.0, ry = 0.0;
    if (j < n) {
      const double2 hj = pos_ld(pos + row_entry(cv, k.N, c, j), k);
      rx = min_image(__dsub_rn(hj.x, h0.x), k.Lx, k.hLx);
      ry = min_image(__dsub_rn(hj.y, h0.y), k.Ly, k.hLy);
    }
    geom_edge(rxp, ryp, rx, ry, acc, per);
    rxp = rx; ryp = ry;
  }
  A = __dmul_rn(0.5, acc); P = per;
}

// |d| >= L/2 decided conservatively on the high word with integer ALU ops (keeps the FP64 pipe
// for arithmetic); the exact minimum image runs only where this fires.
__device__ __forceinline__ unsigned may_wrap(double d, unsigned hi_half) { return (hi_word(d) & 0x7fffffffu) >= hi_half; }

// ---------------------------------------------------------------------------------------------
// rows a2 + a3: vertex forces (Eq. A2-A5) and displacement (Eq. 4, :56).
// Slot convention (R12): in cell c_k = vc[v][k] the CCW neighbours of v are next = vn[v][k],
// prev = vn[v][k+1], so no row search is needed.  With r_k = mi(h_{n_k} - h_v):
//   dA_{c_k}/dh_v = 1/2 (r_k.y - r_{k+1}.y, r_{k+1}.x - r_k.x)        (A4, R3)
//   dP_{c_k}/dh_v = -(rhat_k + rhat_{k+1})                             (A5, R2)
//   F_v = -sum_k [ a_k dA + p_k dP ],  a = 2K_A(A-A0), p = 2K_P(P-P0)  (A2, A3)
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double2 vertex_force(const double2 h, const double2 q0, const double2 q1,
                                                const double2 q2, const CellRec& c0, const CellRec& c1,
                                                const CellRec& c2, const Consts& k) {
  // Explicit rounding intrinsics throughout: the function is instantiated in several kernels
  // (sweep, post-flip move, avm_compute_forces) and must give the same bits in each, so no
  // contraction is left to the compiler.
  double r0x = __dsub_rn(q0.x, h.x), r0y = __dsub_rn(q0.y, h.y), r1x = __dsub_rn(q1.x, h.x), r1y = __dsub_rn(q1.y, h.y),
         r2x = __dsub_rn(q2.x, h.x), r2y = __dsub_rn(q2.y, h.y);
  const unsigned hx = hi_word(k.hLx), hy = hi_word(k.hLy);
  if (may_wrap(r0x, hx) | may_wrap(r1x, hx) | may_wrap(r2x, hx) | may_wrap(r0y, hy) | may_wrap(r1y, hy) | may_wrap(r2y, hy)) {
    r0x = min_image(r0x, k.Lx, k.hLx); r1x = min_image(r1x, k.Lx, k.hLx); r2x = min_image(r2x, k.Lx, k.hLx);
    r0y = min_image(r0y, k.Ly, k.hLy); r1y = min_image(r1y, k.Ly, k.hLy); r2y = min_image(r2y, k.Ly, k.hLy);
  }
  // + kTiny: a zero-length edge gives r * rsqrt = 0, i.e. contributes nothing (R15)
  const double i0 = rsqrt_pos(__fma_rn(r0x, r0x, __fma_rn(r0y, r0y, kTiny)));
  const double i1 = rsqrt_pos(__fma_rn(r1x, r1x, __fma_rn(r1y, r1y, kTiny)));
  const double i2 = rsqrt_pos(__fma_rn(r2x, r2x, __fma_rn(r2y, r2y, kTiny)));
  const double u0x = __dmul_rn(r0x, i0), u0y = __dmul_rn(r0y, i0), u1x = __dmul_rn(r1x, i1), u1y = __dmul_rn(r1y, i1),
               u2x = __dmul_rn(r2x, i2), u2y = __dmul_rn(r2y, i2);
  // cell k uses (next, prev) = (r_k, r_{k+1})
  double sx = __dmul_rn(c0.a, __dsub_rn(r0y, r1y));
  sx = __fma_rn(c1.a, __dsub_rn(r1y, r2y), sx);
  sx = __fma_rn(c2.a, __dsub_rn(r2y, r0y), sx);
  double sy = __dmul_rn(c0.a, __dsub_rn(r1x, r0x));
  sy = __fma_rn(c1.a, __dsub_rn(r2x, r1x), sy);
  sy = __fma_rn(c2.a, __dsub_rn(r0x, r2x), sy);
  double fx = __dmul_rn(-0.5, sx), fy = __dmul_rn(-0.5, sy);
  fx = __fma_rn(c0.p, __dadd_rn(u0x, u1x), fx); fx = __fma_rn(c1.p, __dadd_rn(u1x, u2x), fx); fx = __fma_rn(c2.p, __dadd_rn(u2x, u0x), fx);
  fy = __fma_rn(c0.p, __dadd_rn(u0y, u1y), fy); fy = __fma_rn(c1.p, __dadd_rn(u1y, u2y), fy); fy = __fma_rn(c2.p, __dadd_rn(u2y, u0y), fy);
  return make_double2(fx, fy);
}

// Candidate lists.  List 0 / 1 (the step's list, by step parity) starts at d.cand and holds up to
// k.cap_a = 3N entries; lists 2 / 3 (repeated passes, NEXT-1; allocated only when they are enabled)
// hold up to N entries each behind it.
__device__ __forceinline__ Cand* list_base(const Dev& d, const Consts& k, unsigned list) {
  return d.cand + (list < 2u ? (size_t)0 : (size_t)(list + 1u) * (size_t)k.N);
}
__device__ __forceinline__ unsigned list_cap(const Consts& k, unsigned list) { return list < 2u ? (unsigned)k.cap_a : (unsigned)k.N; }

// ---------------------------------------------------------------------------------------------
// host-side launchers (defined in the .cu files); every launcher returns the number of kernels
// it enqueued so that the API can keep avm_stats.kernel_launches honest.
// ---------------------------------------------------------------------------------------------
int force_move_grid(int V);
// One timestep.  consume_pending: the previous step left its T1 flips pending (they ride in this force/move
// launch); leave_pending: this step leaves its own flips pending (two launches) instead of running t1_flip_kernel.
// obs_partial (optional, one double per observable slot and CTA of the cell pass): the cell pass also reduces the
// observables of the moved tiling (avm_step_observe).
int launch_step(const Dev& d, const Consts& k, unsigned long long step, cudaStream_t s, cudaEvent_t* ev, bool consume_pending,
                bool leave_pending, double* obs_partial = nullptr);
int cell_pass_grid(int N);
int launch_count_short_edges(const Dev& d, const Consts& k, cudaStream_t s);
int persistent_grid(int V, bool per_cell);
int launch_persistent_steps(const Dev& d, const Consts& k, unsigned long long step0, int n_steps, int grid, cudaStream_t s);
int launch_refresh_cells(const Dev& d, const Consts& k, cudaStream_t s);
int launch_t1_reset(const Dev& d, const Consts& k, cudaStream_t s);
int launch_t1_pass_only(const Dev& d, const Consts& k, cudaStream_t s);
int launch_t1_extra_pass(const Dev& d, const Consts& k, unsigned list_prev, unsigned list_new, unsigned stamp, cudaStream_t s);
int launch_t1_release(const Dev& d, const Consts& k, unsigned list, cudaStream_t s);
int launch_t1_debug(const Dev& d, const Consts& k, int* cand_pairs, int* win_pairs, long long capacity, cudaStream_t s);
int launch_compute_forces(const Dev& d, const Consts& k, double2* ap_scratch, double* force_user, double* ap_user, cudaStream_t s);
int launch_energy(const Dev& d, const Consts& k, double* partial, cudaStream_t s);
int launch_philox_words(unsigned long long seed, unsigned long long step, unsigned long long cell0, long long n, uint32_t* out, cudaStream_t s);

// SPV on a fixed triangulation (avm_spv.cu)
int launch_spv_voronoi(const Dev& d, const Consts& k, const double* cell_xy, double* voronoi_user, cudaStream_t s);
int launch_spv_forces(const Dev& d, const Consts& k, const double* cell_xy, double2* g_scratch, double2* force_int, double* force_user,
                      double* sets_user, cudaStream_t s);
int launch_spv_move(const Dev& d, const Consts& k, double* cell_xy, const double2* force_int, double v0, unsigned long long step,
                    cudaStream_t s);
int launch_spv_test(const Dev& d, const Consts& k, const double* cell_xy, unsigned long long* counts, int* flags,
                    unsigned long long step_rel, cudaStream_t s);

struct SortScratch {
  unsigned int* key[2];   // [max(V,N)] each
  int* val[2];            // [max(V,N)]
  unsigned int* hist;     // [256 * n_warps_max]
  int* newidx_v;          // [V] old -> new
  int* newidx_c;          // [N]
  int* order_v;           // [V] new -> old
  int* order_c;           // [N]
};
size_t sort_hist_entries(int n);
// Hilbert re-sort: reads buffer set `a`, writes set `b` (all arrays permuted and re-indexed).
int launch_hilbert_sort(const Dev& a, const Dev& b, const Consts& k, const SortScratch& sc, cudaStream_t s);

}  // namespace avm
