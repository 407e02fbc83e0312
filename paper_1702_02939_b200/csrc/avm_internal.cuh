// avm_internal.cuh — shared declarations of the CUDA path (sm_100a).  Not part of the C ABI.
//
// Notation follows the paper (PAPER.md = /root/reference/PAPER.md): h = vertex position,
// A/P = cell area / perimeter, theta = director angle, cellVertices / vertexNeighbors /
// vertexCellNeighbors = the three flat topology lists of PAPER.md:66.  R-numbers = DESIGN.md.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/avm.h"

namespace avm {

// Per-cell record gathered by the force/move kernel: one 32-byte sector per cell.
//   a  = 2 K_A (A_c - A0)   (Eq. A3 prefactor)
//   p  = 2 K_P (P_c - P0)
//   nx = cos(theta_c), ny = sin(theta_c)   (director)
struct __align__(32) CellRec { double a, p, nx, ny; };

// One eligible T1 candidate (R10), decoded once by t1_mark and reused by t1_flip / t1_reset.
struct __align__(16) Cand {
  int v1, v2;           // v1 = endpoint with the smaller tag
  int k1, k2;           // slot of v2 in v1, slot of v1 in v2
  int cL, cR, cE1, cE2; // the two cells sharing the edge, the two end cells (R12)
  unsigned long long key;  // (tag(v1) << 32) | tag(v2)  (R11)
  unsigned long long pad;
};

struct Counters {
  unsigned int n_short;   // short edges appended this step
  unsigned int n_cand;    // eligible candidates this step
  unsigned int n_win;     // winners (debug hook only)
  unsigned int pad;
  long long t1_short, t1_candidates, t1_flips, t1_blocked, overflow_rejects, error;
  double energy;
};

// Model constants, passed by value to every kernel.
struct Consts {
  int N, V, S;
  double Lx, Ly, hLx, hLy;
  double KA2, KP2, A0, P0;   // KA2 = 2 K_A, KP2 = 2 K_P
  double KA, KP;
  double v0_3, mu, dt;       // v0_3 = v0 / 3 (Eq. 4 with n = 3, R5)
  double amp;                // sqrt(2 Dr dt) (R8)
  double lc, lc2;
  unsigned long long seed;
};

// Pointers into the caller's workspace (current buffer set).
struct Dev {
  double2* pos;       // [V] current positions
  double2* pos_next;  // [V] written by force_move, then swapped
  int* vn;            // [3V] vertexNeighbors
  int* vc;            // [3V] vertexCellNeighbors
  int* cv;            // [N*S] cellVertices (rows), unused = -1
  int* cvn;           // [N] cellVertexNum
  double* theta;      // [N]
  CellRec* rec;       // [N]
  int* vtag;          // [V] user index of each vertex
  int* ctag;          // [N] user index of each cell
  unsigned long long* minkey;  // [N] per-cell minimum candidate key, ~0 when idle
  int2* short_list;   // [3N] short edges found by the detection pass
  Cand* cand;         // [3N]
  Counters* ctr;
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

// Philox4x32-10 (Salmon et al., SC'11; R16).  Counter (c0..c3), key (k0,k1).
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const unsigned int hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
    const unsigned int hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
    c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
    k.x += 0x9E3779B9u; k.y += 0xBB67AE85u;
  }
  return c;
}
__device__ __forceinline__ uint4 philox_for(unsigned long long seed, unsigned long long step,
                                            unsigned long long cell) {
  return philox4x32_10(make_uint4((unsigned)step, (unsigned)(step >> 32), (unsigned)cell, (unsigned)(cell >> 32)),
                       make_uint2((unsigned)seed, (unsigned)(seed >> 32)));
}
// Standard normal from one Philox block: two 52-bit uniforms in (0,1), Box-Muller cosine branch.
__device__ __forceinline__ double director_noise(unsigned long long seed, unsigned long long step,
                                                 unsigned long long cell) {
  const uint4 x = philox_for(seed, step, cell);
  const unsigned long long a = ((unsigned long long)x.y << 32) | x.x;
  const unsigned long long b = ((unsigned long long)x.w << 32) | x.z;
  const double u1 = ((double)(a >> 12) + 0.5) * 2.220446049250313e-16;   // 2^-52
  const double u2 = ((double)(b >> 12) + 0.5) * 2.220446049250313e-16;
  return sqrt(-2.0 * log(u1)) * cospi(2.0 * u2);
}

// Area and perimeter of one cell from its row (Eq. A1 inputs; shoelace with every vertex
// unwrapped relative to the row's first vertex, R14).  Used by the cold paths (T1 flip refresh,
// avm_compute_forces); the per-step pass has its own fused copy.
__device__ __forceinline__ void cell_area_perimeter(const double2* __restrict__ pos, const int* __restrict__ row,
                                                    int n, const Consts& k, double& A, double& P) {
  const double2 h0 = pos[row[0]];
  double rx_prev = 0.0, ry_prev = 0.0, acc = 0.0, per = 0.0;
  for (int j = 1; j <= n; ++j) {
    double rx = 0.0, ry = 0.0;
    if (j < n) {
      const double2 hj = pos[row[j]];
      rx = min_image(hj.x - h0.x, k.Lx, k.hLx);
      ry = min_image(hj.y - h0.y, k.Ly, k.hLy);
    }
    acc += rx_prev * ry - ry_prev * rx;
    const double dx = rx - rx_prev, dy = ry - ry_prev;
    per += sqrt(dx * dx + dy * dy);
    rx_prev = rx; ry_prev = ry;
  }
  A = 0.5 * acc; P = per;
}

// ---------------------------------------------------------------------------------------------
// host-side launchers (defined in the .cu files); every launcher returns the number of kernels
// it enqueued so that the API can keep avm_stats.kernel_launches honest.
// ---------------------------------------------------------------------------------------------
int launch_step(const Dev& d, const Consts& k, unsigned long long step, cudaStream_t s, cudaEvent_t* ev = nullptr);
int launch_refresh_cells(const Dev& d, const Consts& k, cudaStream_t s);
int launch_t1_pass_only(const Dev& d, const Consts& k, cudaStream_t s);
int launch_t1_debug(const Dev& d, const Consts& k, int* cand_pairs, int* win_pairs, long long capacity, cudaStream_t s);
int launch_compute_forces(const Dev& d, const Consts& k, double2* ap_scratch, double* force_user, double* ap_user, cudaStream_t s);
int launch_energy(const Dev& d, const Consts& k, double* partial, cudaStream_t s);
int launch_philox_words(unsigned long long seed, unsigned long long step, unsigned long long cell0, long long n, uint32_t* out, cudaStream_t s);

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
