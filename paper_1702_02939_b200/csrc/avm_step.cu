// avm_step.cu — the per-timestep kernels of the AVM hot path for sm_100a.
//
// Paper order of one step (PAPER.md:62-64 §II.B, :104-108 §II.D; R6):
//   geometry -> forces -> move vertices -> rotate directors -> T1 test/update.
// Kernel schedule used here:
//   force_move   (thread/vertex)  rows a2+a3: F_v from the 3 incident cells' cached (a,p) records
//                                  and the 3 neighbour positions, Euler step of Eq. 4, wrap.
//   cell_update  (thread/cell)    rows a4+a1+a5+a6: director noise, then area/perimeter of the MOVED
//                                  tiling (= the geometry the next step's forces need); edges found
//                                  shorter than l_c are tested for eligibility by the detecting
//                                  thread, appended to the candidate list and their key is
//                                  atomicMin-ed into the four cells (conflict rule, marking half).
//   T1 flips     (4 lanes/candidate) rows a6+a7 (t1_flip_quads): a candidate whose key is the minimum
//                                  on all four of its cells flips; each of the four lanes rewrites
//                                  one cell row and refreshes that cell's cached geometry.
//                                  Two-launch schedule (large systems): run by a few "flipper"
//                                  warps inside the NEXT step's force_move launch while the other
//                                  warps sweep.  Three-launch schedule: t1_flip_kernel.
//   repeated T1 passes (NEXT-1)    t1_release / t1_local_detect / t1_flip per extra pass.
// Geometry is thus evaluated once per step on the positions the forces of the following step
// act on; after a flip the records of its four cells are refreshed in place, so every force is
// computed from the geometry of the current topology exactly as in the paper's cycle.
#include <cstdio>
#include <cstdlib>
#include <cooperative_groups.h>
#include <utility>
#include "avm_internal.cuh"

namespace avm {
namespace cg = cooperative_groups;

#ifndef AVM_VERTEX_BLOCK
#define AVM_VERTEX_BLOCK 256
#endif
static constexpr int kVertexBlock = AVM_VERTEX_BLOCK;
#ifndef AVM_CELL_BLOCK
#define AVM_CELL_BLOCK 64
#endif
static constexpr int kCellBlock = AVM_CELL_BLOCK;
static constexpr int kT1Block = 128;
#ifndef AVM_T1_GRID
#define AVM_T1_GRID (148 * 3)      // CTAs of the T1 kernels (166 registers: three CTAs of 128 per SM; measured against 148 x 2: -0.5 us/step in the burst and at configs[2])
#endif
static constexpr int kT1Grid = AVM_T1_GRID;
static constexpr unsigned kFull = 0xffffffffu;

// tuning knobs (compile-time; the defaults are the measured best, profiles/)
#ifndef AVM_FM_PF
#define AVM_FM_PF 1        // force_move: L2 prefetch distance in grid sweeps (0 = off)
#endif
#ifndef AVM_PDL
#define AVM_PDL 1          // chain the step's kernels with programmatic dependent launch
#endif
#ifndef AVM_CU_MINB
#define AVM_CU_MINB 16     // cell pass: resident CTAs per SM asked of the compiler (64 registers; CTAs of 64 threads x 16 per SM: a CTA that holds a T1-marking thread keeps fewer idle warps resident; measured against 128 x 8: -0.3 us steady, -0.8 us in the burst, -2 us at N = 4M)
#endif
#ifndef AVM_FM_MINB
#define AVM_FM_MINB 3      // force_move: minimum resident CTAs per SM asked of the compiler
#endif
#ifndef AVM_TEST_SKEW
#define AVM_TEST_SKEW 0     // test builds: hold back the sweepers (1) or the flippers (2) of the fused launch
#endif
#ifndef AVM_FM_REGPF
#define AVM_FM_REGPF 0     // force_move: keep the next vertex's streaming loads in registers (measured: the L2 prefetch does better)
#endif

// Programmatic dependent launch (sm_90+): the three kernels of a step form a chain on one stream.
// Each kernel lets its successor's CTAs be scheduled as soon as all of its own CTAs have started
// (pdl_launch_dependents) and itself waits for the predecessor's completion and memory flush
// before it touches anything (pdl_wait), so launch latency and the drain of the last wave are
// hidden while the ordering of plain stream semantics is kept.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;"); }

__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// ---- cache-hinted loads -------------------------------------------------------------------------
// Pure streams (index lists, tags) are read once per step: evict-first so that they do not push
// the re-used arrays (positions, cell records) out of L1/L2.
__device__ __forceinline__ int ld_stream(const int* p) { return __ldcs(p); }
__device__ __forceinline__ int4 ld_stream(const int4* p) { return __ldcs(p); }
__device__ __forceinline__ double ld_stream(const double* p) { return __ldcs(p); }
// one record with a single load: 256 bits in the fp64 build (LDG.E.256, sm_100), 128 bits (four floats) in the mixed build
#if AVM_MIXED
__device__ __forceinline__ CellRec ld_rec(const rec_t* p) { return rec_unpack(__ldg(reinterpret_cast<const float4*>(p))); }
__device__ __forceinline__ void st_rec(rec_t* p, const CellRec& r) {
  *reinterpret_cast<float4*>(p) = make_float4((float)r.a, (float)r.p, (float)r.nx, (float)r.ny);
}
#else
__device__ __forceinline__ CellRec ld_rec(const CellRec* p) {
  CellRec r;
  asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(r.a), "=d"(r.p), "=d"(r.nx), "=d"(r.ny) : "l"(p));
  return r;
}
__device__ __forceinline__ void st_rec(CellRec* p, const CellRec& r) {
  asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(r.a), "d"(r.p), "d"(r.nx), "d"(r.ny) : "memory");
}
#endif
struct VertexIn { double2 h; int n0, n1, n2, c0, c1, c2; };
__device__ __forceinline__ VertexIn load_vertex(const Dev& d, const Consts& k, int v) {
  VertexIn in;
  in.h = pos_ldg(d.pos + v, k);
  in.n0 = ld_stream(d.vn + v); in.n1 = ld_stream(d.vn + k.Vs + v); in.n2 = ld_stream(d.vn + 2 * k.Vs + v);
  in.c0 = ld_stream(d.vc + v); in.c1 = ld_stream(d.vc + k.Vs + v); in.c2 = ld_stream(d.vc + 2 * k.Vs + v);
  return in;
}

// Eq. 4: dh/dt = mu F + (v0/3) sum of the three unit directors (R5), directors of the start of
// the step (R7); explicit Euler; wrap into the box (R13).
// kMover: the caller is a post-flip mover of the two-launch schedule (mover_unit).  Those move a vertex once per
// candidate whose cells hold it, with the same inputs and the same result, so everything here is idempotent except
// the image count of the mean-square displacement: the first mover to exchange this step's stamp applies it, the
// others find the stamp and leave the count alone.  Every other caller moves each vertex exactly once per step.
__device__ __forceinline__ bool img_claim(const Dev& d, int tag, unsigned long long step) {
  return atomicExch(d.img_stamp + tag, step + 1ull) != step + 1ull;
}
template <bool kMover = false>
__device__ __forceinline__ void move_vertex(const Dev& d, const Consts& k, int v, const double2 h, const double2 q0,
                                            const double2 q1, const double2 q2, const CellRec& c0, const CellRec& c1,
                                            const CellRec& c2, const unsigned long long step = 0ull) {
  const double2 f = vertex_force(h, q0, q1, q2, c0, c1, c2, k);
  const double vx = __fma_rn(k.mu, f.x, __dmul_rn(k.v0_3, __dadd_rn(__dadd_rn(c0.nx, c1.nx), c2.nx)));
  const double vy = __fma_rn(k.mu, f.y, __dmul_rn(k.v0_3, __dadd_rn(__dadd_rn(c0.ny, c1.ny), c2.ny)));
  double x = __fma_rn(k.dt, vx, h.x), y = __fma_rn(k.dt, vy, h.y);
  // negative, >= L (conservatively) and non-finite values all have a large unsigned high word
#if AVM_MIXED
  int ix = 0, iy = 0;
  if ((hi_word(x) >= hi_word(k.Lx)) | (hi_word(y) >= hi_word(k.Ly))) {
    x = wrap_box_count(x, k.Lx, ix); y = wrap_box_count(y, k.Ly, iy);
    if (!(isfinite(x) && isfinite(y))) atomicOr((unsigned long long*)&d.ctr->error, 1ull);
  }
  const pos_t pk = pos_pack(make_double2(x, y), k);
  if (pk.x == 0u && x > k.hLx) ++ix;    // rounded up to the box length: the grid point is the origin of the next image
  if (pk.y == 0u && y > k.hLy) ++iy;
  d.pos_next[v] = pk;
  if (ix | iy) {
    const int tag = d.vtag[v];
    if (!kMover || img_claim(d, tag, step)) {
      int2* im = d.img + tag;
      int2 c = *im; c.x += ix; c.y += iy; *im = c;
    }
  }
#else
  if ((hi_word(x) >= hi_word(k.Lx)) | (hi_word(y) >= hi_word(k.Ly))) {
    int ix = 0, iy = 0;
    x = wrap_box_count(x, k.Lx, ix); y = wrap_box_count(y, k.Ly, iy);
    if (!(isfinite(x) && isfinite(y))) atomicOr((unsigned long long*)&d.ctr->error, 1ull);
    if (ix | iy) {                      // the vertex left through the boundary: keep its unwrapped position (MSD)
      const int tag = d.vtag[v];
      if (!kMover || img_claim(d, tag, step)) {
        int2* im = d.img + tag;
        int2 c = *im; c.x += ix; c.y += iy; *im = c;
      }
    }
  }
  d.pos_next[v] = make_double2(x, y);
#endif
}

// the same vertex update with every input read from L2 (after another warp of this launch
// rewrote the neighbourhood: L1 may hold stale lines)
// (one-CTA persistent kernel: plain cached loads, see cu_stream)
// (inlined into the persistent kernel: cfg0 2.24 -> 2.00 us/step, cfg1 7.5 -> 6.9)
#ifndef AVM_PERS_ATTR
#define AVM_PERS_ATTR __forceinline__
#endif
__device__ AVM_PERS_ATTR void move_vertex_plain(const Dev& d, const Consts& k, int v) {
  const double2 h = pos_ld(d.pos + v, k);
  double2 q[3];
  CellRec c[3];
#pragma unroll
  for (int s = 0; s < 3; ++s) {
    q[s] = pos_ld(d.pos + d.vn[s * k.Vs + v], k);
    c[s] = rec_ld_plain(d.rec + d.vc[s * k.Vs + v]);
  }
  move_vertex(d, k, v, h, q[0], q[1], q[2], c[0], c[1], c[2]);
}
// helpers of the fused launch: inlined (measured -0.2 us/step against calls; the flip itself stays a call there: inlined
// into the 80-register kernel it costs the sweep 3.7 us)
#ifndef AVM_FUSED_ATTR
#define AVM_FUSED_ATTR __forceinline__
#endif
template <bool kMover = false>
__device__ AVM_FUSED_ATTR void move_vertex_coherent(const Dev& d, const Consts& k, int v, const unsigned long long step = 0ull) {
  const double2 h = pos_ldcg(d.pos + v, k);
  double2 q[3];
  CellRec c[3];
#pragma unroll
  for (int s = 0; s < 3; ++s) {
    q[s] = pos_ldcg(d.pos + __ldcg(d.vn + s * k.Vs + v), k);
    c[s] = rec_ldcg(d.rec + __ldcg(d.vc + s * k.Vs + v));
  }
  move_vertex<kMover>(d, k, v, h, q[0], q[1], q[2], c[0], c[1], c[2], step);
}

// The host chooses the schedule of later steps from the T1 load (avm_api.cu: leave_flips_pending), which it
// reads from a mapped host word.  A store to host memory must be flushed over PCIe before the kernel
// can complete (measured: up to 0.7 us per step), so the word is only written when the load crosses the
// threshold the host compares it with.
__device__ __forceinline__ void report_t1_load(const Dev& d, const unsigned n) {
  const unsigned last = d.ctr->fb_last;
  if ((n > (unsigned)AVM_FUSED_MAX_CANDIDATES) != (last > (unsigned)AVM_FUSED_MAX_CANDIDATES)) {
    d.ctr->fb_last = n;
    *d.feedback = n;
  }
}

__device__ AVM_PERS_ATTR void move_two_coherent(const Dev& d, const Consts& k, int va, int vb) {
  const double2 ha = pos_ldcg(d.pos + va, k), hb = pos_ldcg(d.pos + vb, k);
  int na[3], nb[3], ca[3], cb[3];
#pragma unroll
  for (int s = 0; s < 3; ++s) {
    na[s] = __ldcg(d.vn + s * k.Vs + va); nb[s] = __ldcg(d.vn + s * k.Vs + vb);
    ca[s] = __ldcg(d.vc + s * k.Vs + va); cb[s] = __ldcg(d.vc + s * k.Vs + vb);
  }
  double2 qa[3], qb[3];
  CellRec ra[3], rb[3];
#pragma unroll
  for (int s = 0; s < 3; ++s) {
    qa[s] = pos_ldcg(d.pos + na[s], k); qb[s] = pos_ldcg(d.pos + nb[s], k);
    ra[s] = rec_ldcg(d.rec + ca[s]); rb[s] = rec_ldcg(d.rec + cb[s]);
  }
  move_vertex(d, k, va, ha, qa[0], qa[1], qa[2], ra[0], ra[1], ra[2]);
  move_vertex(d, k, vb, hb, qb[0], qb[1], qb[2], rb[0], rb[1], rb[2]);
}

__device__ __forceinline__ unsigned int ld_volatile(const unsigned int* p) {
  unsigned int x;
  asm volatile("ld.volatile.global.u32 %0, [%1];" : "=r"(x) : "l"(p) : "memory");
  return x;
}

__device__ __noinline__ unsigned t1_flip_quads(const Dev& d, const Consts& k, const Cand* __restrict__ list, unsigned base,
                                               unsigned n, const int lane);
template <int kR>
__device__ __forceinline__ unsigned t1_flip_quads_impl(const Dev& d, const Consts& k, const Cand* __restrict__ list,
                                                       const unsigned base, const unsigned n, const int lane_in,
                                                       const int4* __restrict__ pre = nullptr);
#ifndef AVM_PERS_FLIP_INLINE
#define AVM_PERS_FLIP_INLINE 1    // persistent kernel: the flip inlined too (cfg0 2.00 -> 1.95 us/step, cfg1 6.9 -> 6.7)
#endif
#ifndef AVM_FUSED_FLIP_INLINE
#define AVM_FUSED_FLIP_INLINE 0
#endif

// The sweep of one thread over vertices first, first + step_v, ...  kSkipDirty: vertices flagged
// in `dirty` (read-only for this whole launch) are left to the dirty pass below.
template <bool kSkipDirty>
__device__ __forceinline__ void sweep(const Dev& d, const Consts& k, const unsigned int* __restrict__ dirty, const int first,
                                      const int step_v, const int lane) {
  if (first >= k.V) return;
  int v = first;
  VertexIn in = load_vertex(d, k, v);
  unsigned dw = kSkipDirty ? __ldg(dirty + (v >> 5)) : 0u;
  for (;;) {
    if (AVM_FM_PF) {
      // pull the contiguous streams of a later sweep into L2: positions, both index lists and the
      // cell records around v/2 (cells and vertices share the Hilbert order, so this window also
      // holds most of that sweep's gather targets)
      const long long vb = (long long)(v - lane) + (long long)AVM_FM_PF * step_v;
      if (vb + 32 <= k.V) {
        const char* a = nullptr;
        if (lane < 4) a = reinterpret_cast<const char*>(d.pos + vb) + 128 * lane;
        else if (lane < 7) a = reinterpret_cast<const char*>(d.vn + (size_t)(lane - 4) * k.Vs + vb);
        else if (lane < 10) a = reinterpret_cast<const char*>(d.vc + (size_t)(lane - 7) * k.Vs + vb);
        else if (lane < 14) a = reinterpret_cast<const char*>(d.rec + (vb >> 1)) + 128 * (lane - 10);
        if (a) prefetch_l2(a);
      }
    }
    const bool skip = kSkipDirty && ((dw >> (v & 31)) & 1u);
    const int vnext = v + step_v;
    if (!skip) {
      const double2 q0 = pos_ldg(d.pos + in.n0, k), q1 = pos_ldg(d.pos + in.n1, k), q2 = pos_ldg(d.pos + in.n2, k);
      const CellRec c0 = ld_rec(d.rec + in.c0), c1 = ld_rec(d.rec + in.c1), c2 = ld_rec(d.rec + in.c2);
      const double2 h = in.h;
      if (AVM_FM_REGPF && vnext < k.V) { in = load_vertex(d, k, vnext); if (kSkipDirty) dw = __ldg(dirty + (vnext >> 5)); }
      move_vertex(d, k, v, h, q0, q1, q2, c0, c1, c2);
    } else if (AVM_FM_REGPF && vnext < k.V) {
      in = load_vertex(d, k, vnext);
      dw = __ldg(dirty + (vnext >> 5));
    }
    if (vnext >= k.V) break;
    v = vnext;
    if (!AVM_FM_REGPF) { in = load_vertex(d, k, v); if (kSkipDirty) dw = __ldg(dirty + (v >> 5)); }
  }
}

// Rows a6 + a7 of the previous step inside the fused force_move launch.
//   flips : candidates are CLAIMED eight at a time with an atomic counter and decided / flipped by
//           t1_flip_quads (four lanes per candidate).
//   wait  : until every candidate has been decided (flip_done == prev).
//   moves : one unit per candidate, claimed likewise: the vertices of its four cells (exactly the
//           vertices whose inputs a flip can rewrite; the sweep skipped them) are moved now and
//           the cells' minimum keys are released.
// A few "flipper" warps do nothing else, so with few candidates all of this runs in the shadow of
// the sweep; with many candidates every warp also claims what is left once its share of the
// sweep is done.  Work is claimed, so a candidate always belongs to a warp that is running: the
// wait can never depend on a CTA that has not been scheduled (no co-residency assumption; in the
// few-candidate mode the waiting flipper warps claim what is still unclaimed after ~4 us).
// The bitmap of flagged vertices is read-only for the whole launch (the cell pass of the previous
// step wrote it, the cell pass of this step clears it), so the sweep's decision to skip a vertex
// never changes while flips are in flight.
// first: a batch already claimed for this warp (by its CTA), or >= prev for none
__device__ AVM_FUSED_ATTR void flipper_flips(const Dev& d, const Consts& k, const unsigned prev, const int lane, const unsigned first) {
  unsigned mine = 0, flips = 0;
  unsigned i = first;
  for (;;) {
    if (i >= prev) {
      const unsigned nc = ld_volatile(&d.ctr->next_cand);
      if (nc >= prev) break;        // nothing left: no atomic
      if (lane == 0) i = atomicAdd(&d.ctr->next_cand, 8u);
      i = __shfl_sync(kFull, i, 0);
      if (i >= prev) break;
    }
    flips += (AVM_FUSED_FLIP_INLINE && k.S <= 16) ? t1_flip_quads_impl<16>(d, k, d.cand, i, prev, lane) : t1_flip_quads(d, k, d.cand, i, prev, lane);
    mine += min(8u, prev - i);
    i = prev;
  }
  if (mine) {
    __threadfence();
    __syncwarp();
    if (lane == 0) {
      if (flips) atomicAdd((unsigned long long*)&d.ctr->t1_flips, (unsigned long long)flips);
      if (mine - flips) atomicAdd((unsigned long long*)&d.ctr->t1_blocked, (unsigned long long)(mine - flips));
      atomicAdd(&d.ctr->flip_done, mine);
    }
  }
}

// One unit of post-flip work = one candidate (few-candidate mode): every vertex of the (post-flip)
// rows of its four cells is moved, with loads that bypass L1, and the cells' minimum keys go back
// to idle (row a6).  Units are assigned statically: nothing ever waits for a unit.
// Lanes = 4 cells x 8 row entries per pass (96 % of the cells need one pass); a vertex that sits
// in several of the four rows is moved by the lowest lane holding it.  A vertex shared with
// another candidate's cells (or met again in a later pass of a long row) is moved twice, with the same inputs
// and the same result; its image count is applied once (img_claim).
__device__ AVM_FUSED_ATTR void mover_unit(const Dev& d, const Consts& k, const unsigned i, const int lane, const unsigned long long step) {
  const int t = lane >> 3, j8 = lane & 7;
  const int4 q = __ldcg(reinterpret_cast<const int4*>(d.cand + i) + 1);   // (cL, cR, cE1, cE2)
  const int cell = t == 0 ? q.x : t == 1 ? q.y : t == 2 ? q.z : q.w;
  // entry j8 is loaded whatever the row length is (padding repeats entry 0): no dependent load
  const int n = __ldcg(d.cvn + cell);
  int u = __ldcg(reinterpret_cast<const int*>(d.cv + (size_t)(j8 >> 2) * k.N + cell) + (j8 & 3));
  int nmax = max(n, __shfl_xor_sync(kFull, n, 8));
  nmax = max(nmax, __shfl_xor_sync(kFull, nmax, 16));
  for (int j0 = 0; j0 < nmax; j0 += 8) {
    const int j = j0 + j8;
    if (j0 > 0 && j < n) u = __ldcg(reinterpret_cast<const int*>(d.cv + (size_t)(j >> 2) * k.N + cell) + (j & 3));
    const int uu = j < n ? u : -1 - lane;                                   // inactive lanes match nobody
    const unsigned same = __match_any_sync(kFull, uu);
    if (j < n && __ffs(same) - 1 == lane) move_vertex_coherent<true>(d, k, u, step);
  }
  if (lane < 4) d.minkey[lane == 0 ? q.x : lane == 1 ? q.y : lane == 2 ? q.z : q.w] = ~0ull;
}

// minimum keys of candidates [i0, i1) back to idle (row a6), thread per candidate
__device__ __forceinline__ void release_minkeys(const Dev& d, const unsigned i0, const unsigned i1, const unsigned step, const unsigned first) {
  for (unsigned i = i0 + first; i < i1; i += step) {
    const int4 q = __ldcg(reinterpret_cast<const int4*>(d.cand + i) + 1);   // (cL, cR, cE1, cE2)
    d.minkey[q.x] = ~0ull; d.minkey[q.y] = ~0ull; d.minkey[q.z] = ~0ull; d.minkey[q.w] = ~0ull;
  }
}

// Persistent grid-stride kernel (thread per vertex, rows a2 + a3).
//
// kFused also carries rows a6 + a7 of the PREVIOUS step (above): a few warps decide and flip that
// step's candidates while all other warps already move vertices.  A vertex whose inputs a flip may
// rewrite has its bit set in the bitmap; the sweep skips it and the dirty pass moves it once every
// candidate has been decided.  The latency-bound flips thus overlap the gather-bound sweep and
// the step needs no third launch.
#ifndef AVM_LIGHT_MAX
#define AVM_LIGHT_MAX 1024      // up to this many candidates: one dedicated flipper warp per candidate (measured at N = 1M: 256, 512, 1024, 2048)
#endif
template <bool kFused>
__global__ void __launch_bounds__(kVertexBlock, AVM_FM_MINB)
force_move_kernel(const __grid_constant__ Dev d, const __grid_constant__ Consts k, const unsigned long long step) {
  const unsigned parity = (unsigned)(step & 1ull);
  pdl_launch_dependents();
  pdl_wait();
  const int tid = blockIdx.x * kVertexBlock + threadIdx.x;
  const int stride = gridDim.x * kVertexBlock;
  const int lane = threadIdx.x & 31;
  const unsigned prev = min(d.ctr->n_cand[parity ^ 1u], (unsigned)k.cap_a);
  const unsigned gwarp = (unsigned)tid >> 5, nwarps = (unsigned)stride >> 5;
  if (tid == 0) { d.ctr->n_cand[parity] = 0; if (kFused) report_t1_load(d, prev); }   // whoever applies a list reports its length
  if (kFused) {
    if (prev == 0u) { sweep<false>(d, k, nullptr, tid, stride, lane); return; }
    if (tid == 0) atomicAdd((unsigned long long*)&d.ctr->t1_candidates, (unsigned long long)prev);
    const unsigned int* __restrict__ dirty = d.dirty + (size_t)(parity ^ 1u) * (size_t)k.nw;
    if (prev <= AVM_LIGHT_MAX && 3u * prev <= nwarps) {      // (a small grid must keep most of its warps for the sweep)
      // few candidates: one dedicated warp per candidate (warp 0 of the first CTAs, then warp 1, ...:
      // consecutive CTAs sit on different SMs) flips it, waits for all decisions and moves the
      // vertices of its cells, all in the shadow of the sweep; every other warp only sweeps
      const unsigned wib = threadIdx.x >> 5, nb = gridDim.x;
      const unsigned fid = wib * nb + blockIdx.x;                          // flipper id of this warp, if < prev
      const unsigned full = prev / nb, rest = prev % nb;                   // warps 0..full-1 of every CTA, warp `full` of `rest` CTAs
#if AVM_TEST_SKEW == 1 || AVM_TEST_SKEW == 2
      // Test builds only (tests/test_gpu_skew.py): one side of the launch is held back for tens of microseconds so
      // that the other finishes first.  1: the sweepers start after the flips and the movers are long done;
      // 2: the flippers start after the sweep is long over.  Results must not depend on it.
      // (3, below: every other mover starts 30 us after the rest, so that a vertex two movers share is moved at two
      // clearly different times.)
      if ((AVM_TEST_SKEW == 1) != (fid < prev)) {
        unsigned long long t0, t1;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
        do { __nanosleep(1000); asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1)); } while (t1 - t0 < (AVM_TEST_SKEW == 1 ? 40000ull : 80000ull));
      }
#endif
      if (fid < prev) {
        // The first prev/8 of them claim the flips at once.  The others wait for the decisions, and a waiting warp that
        // has polled for ~4 us tries to claim too: a batch still unclaimed by then belongs to a warp that is not
        // running (a CTA not yet resident: a shared GPU, MPS), so the wait never depends on co-residency.
        bool claim = fid * 8u < prev;
        for (unsigned polls = 0;;) {
          if (claim) { flipper_flips(d, k, prev, lane, prev); claim = false; }
          if (ld_volatile(&d.ctr->flip_done) >= prev) break;
          __nanosleep(64);
          if (++polls == 64u) { polls = 0; claim = true; }
        }
        __threadfence();
#if AVM_TEST_SKEW == 3
        if (fid & 1u) {
          unsigned long long t0, t1;
          asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
          do { __nanosleep(1000); asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1)); } while (t1 - t0 < 30000ull);
        }
#endif
        mover_unit(d, k, fid, lane, step);
      } else {
        const unsigned before = blockIdx.x * full + min(blockIdx.x, rest) + min(wib, full) + (wib > full && blockIdx.x < rest ? 1u : 0u);
        sweep<true>(d, k, dirty, (int)((gwarp - before) * 32u) + lane, (int)((nwarps - prev) * 32u), lane);
      }
    } else {
      // many candidates (the burst after a random start, T1-heavy regimes): the flips come first,
      // claimed by all warps while the SMs are quiet (under the sweep's load every dependent access
      // of a flip takes ~3x longer, and a warp that flips would start a static share of the sweep
      // late and finish last); when every candidate has been decided, a plain sweep moves all vertices
      __shared__ unsigned s_first;
      if (threadIdx.x == 0) s_first = atomicAdd(&d.ctr->next_cand, 8u * (kVertexBlock / 32));   // one claim per CTA
      __syncthreads();
      flipper_flips(d, k, prev, lane, s_first + 8u * (threadIdx.x >> 5));
      while (ld_volatile(&d.ctr->flip_done) < prev) __nanosleep(32);
      __threadfence();
      release_minkeys(d, 0u, prev, (unsigned)stride, (unsigned)tid);       // every decision has been taken (row a6)
      sweep<false>(d, k, nullptr, tid, stride, lane);
    }
  } else {
    // the previous step's T1 candidates are done: clear their cells' minimum keys (row a6)
    for (unsigned i = tid; i < prev; i += stride) {
      const Cand c = d.cand[i];
      d.minkey[c.cL] = ~0ull; d.minkey[c.cR] = ~0ull; d.minkey[c.cE1] = ~0ull; d.minkey[c.cE2] = ~0ull;
    }
    sweep<false>(d, k, nullptr, tid, stride, lane);
  }
}

// ---------------------------------------------------------------------------------------------
// rows a5 (eligibility, R10) + a6 (marking half of the conflict rule, R11) for ONE short edge,
// run by the thread that found it.  (va, vb) are current vertex indices.  Cold path.
// ---------------------------------------------------------------------------------------------
// mode: kMarkFirstPass = the step's detection on the moved positions (counts t1_short /
// overflow_rejects, flags the dirty bitmap of the fused schedule); kMarkRepeatedPass = a repeated
// pass of NEXT-1 (no statistics, but the sticky overflow bit is still raised);
// kMarkSilent = the debug hook (no side effects beyond the list and the minimum keys).
enum : int { kMarkSilent = 0, kMarkFirstPass = 1, kMarkRepeatedPass = 2 };
// (inlined everywhere: a call from the cell pass, even one that is never taken, costs that pass a stack frame, the
// ABI's register partition and generic loads of the by-reference parameter structs: measured 2 us per step)
__device__ __forceinline__ void t1_mark_edge(const Dev& d, const Consts& k, int va, int vb, unsigned parity, const int mode) {
  const bool count_stats = mode == kMarkFirstPass;
  // The marking thread delays the end of the cell pass when it sits in the last wave, so its
  // loads are issued in two batches of independent loads instead of a chain of five.
  // ---- batch 1: everything known from (va, vb) ----
  const double2 ha = pos_ld(d.pos + va, k), hb = pos_ld(d.pos + vb, k);
  const unsigned int ta = (unsigned int)d.vtag[va], tb = (unsigned int)d.vtag[vb];
  int na[3], nb[3], ca[3], cb[3];
#pragma unroll
  for (int s = 0; s < 3; ++s) {
    na[s] = d.vn[s * k.Vs + va]; nb[s] = d.vn[s * k.Vs + vb];
    ca[s] = d.vc[s * k.Vs + va]; cb[s] = d.vc[s * k.Vs + vb];
  }
  // canonical test (R9): strict l < l_c on the minimum-image separation of the two endpoints
  const double dx = min_image(hb.x - ha.x, k.Lx, k.hLx), dy = min_image(hb.y - ha.y, k.Ly, k.hLy);
  if (!(dx * dx + dy * dy < k.lc2)) return;
  if (count_stats) atomicAdd((unsigned long long*)&d.ctr->t1_short, 1ull);
  const bool sw = ta > tb;                    // v1 = endpoint with the smaller tag
  const int v1 = sw ? vb : va, v2 = sw ? va : vb;
  const unsigned int t1 = sw ? tb : ta, t2 = sw ? ta : tb;
  int nb1[3], nb2[3], vc1[3], vc2[3];
#pragma unroll
  for (int s = 0; s < 3; ++s) { nb1[s] = sw ? nb[s] : na[s]; nb2[s] = sw ? na[s] : nb[s]; vc1[s] = sw ? cb[s] : ca[s]; vc2[s] = sw ? ca[s] : cb[s]; }
  const int k1 = nb1[0] == v2 ? 0 : nb1[1] == v2 ? 1 : 2, k2 = nb2[0] == v1 ? 0 : nb2[1] == v1 ? 1 : 2;
  // cyclic from the partner's slot the cells of u are (C0, C1, C2); C0 is left of u -> partner
  const int cL = k1 == 0 ? vc1[0] : k1 == 1 ? vc1[1] : vc1[2], cE1 = k1 == 0 ? vc1[1] : k1 == 1 ? vc1[2] : vc1[0];
  const int cR = k2 == 0 ? vc2[0] : k2 == 1 ? vc2[1] : vc2[2], cE2 = k2 == 0 ? vc2[1] : k2 == 1 ? vc2[2] : vc2[0];
  const bool distinct = cL != cR && cL != cE1 && cL != cE2 && cR != cE1 && cR != cE2 && cE1 != cE2;
  if (!distinct) return;
  // the flip's outer vertices, decoded here so that the flip needs no dependent loads
  const int x1 = k1 == 0 ? nb1[1] : k1 == 1 ? nb1[2] : nb1[0], y1 = k1 == 0 ? nb1[2] : k1 == 1 ? nb1[0] : nb1[1];
  const int x2 = k2 == 0 ? nb2[1] : k2 == 1 ? nb2[2] : nb2[0], y2 = k2 == 0 ? nb2[2] : k2 == 1 ? nb2[0] : nb2[1];
  // ---- batch 2: everything known from the four cells and the outer vertices ----
  const int quad[4] = {cL, cR, cE1, cE2};
  int nq[4];
  int4 q[4][2];
  const bool flag = count_stats && k.flag_dirty;     // the rows are only needed to flag their vertices
#pragma unroll
  for (int t = 0; t < 4; ++t) {
    nq[t] = d.cvn[quad[t]];
    q[t][0] = q[t][1] = make_int4(0, 0, 0, 0);
    if (flag) { q[t][0] = d.cv[quad[t]]; q[t][1] = d.cv[(size_t)k.N + quad[t]]; }
  }
  const int x1s1 = d.vn[k.Vs + x1], x1s2 = d.vn[2 * k.Vs + x1], x2s1 = d.vn[k.Vs + x2], x2s2 = d.vn[2 * k.Vs + x2];
  if (!(nq[0] > 3 && nq[1] > 3)) return;                       // no 2-gons (T2 absent)
  if (!(nq[2] < k.S && nq[3] < k.S)) {                         // row would exceed the stride
    if (count_stats) atomicAdd((unsigned long long*)&d.ctr->overflow_rejects, 1ull);
    if (mode != kMarkSilent) atomicOr((unsigned long long*)&d.ctr->error, 2ull);
    return;
  }
  Cand cd;
  cd.v1 = v1; cd.v2 = v2; cd.k1 = k1; cd.k2 = k2;
  cd.cL = cL; cd.cR = cR; cd.cE1 = cE1; cd.cE2 = cE2;
  cd.key = ((unsigned long long)t1 << 32) | t2;
  cd.x1 = x1; cd.y1 = y1; cd.x2 = x2; cd.y2 = y2;
  // slots of v1 in x1 and of v2 in x2 (2 bits each) and the vertex counts of the four cells (one byte each): a
  // winner owns its four cells (R11), so the counts still hold when it flips and the flip need not load them
  cd.sx1 = (x1s1 == v1 ? 1 : x1s2 == v1 ? 2 : 0) | ((x2s1 == v2 ? 1 : x2s2 == v2 ? 2 : 0) << 2);
  cd.sx2 = nq[0] | (nq[1] << 8) | (nq[2] << 16) | (nq[3] << 24);
  const unsigned int slot = atomicAdd(&d.ctr->n_cand[parity], 1u);
  if (slot >= list_cap(k, parity)) {          // cannot happen for a tiling (<= 3N edges; N per repeated pass)
    atomicOr((unsigned long long*)&d.ctr->error, 8ull);
    return;
  }
  list_base(d, k, parity)[slot] = cd;
  atomicMin(&d.minkey[cL], cd.key);
  atomicMin(&d.minkey[cR], cd.key);
  atomicMin(&d.minkey[cE1], cd.key);
  atomicMin(&d.minkey[cE2], cd.key);
  // Everything a flip of this edge would write, and everything that reads it in the next
  // force/move pass, belongs to a vertex of these four cells: flag them, so that force_move can
  // run the flips while the untouched vertices already move.
  if (flag) {
    unsigned int* __restrict__ dirty = d.dirty + (size_t)parity * (size_t)k.nw;   // this step's bitmap
#pragma unroll
    for (int t = 0; t < 4; ++t) {
      const int e[8] = {q[t][0].x, q[t][0].y, q[t][0].z, q[t][0].w, q[t][1].x, q[t][1].y, q[t][1].z, q[t][1].w};
#pragma unroll
      for (int j = 0; j < 8; ++j) atomicOr(&dirty[e[j] >> 5], 1u << (e[j] & 31));   // padding repeats entry 0
      for (int j = 8; j < nq[t]; ++j) {
        const int u = row_entry(d.cv, k.N, quad[t], j);
        atomicOr(&dirty[u >> 5], 1u << (u & 31));
      }
    }
  }
}

// The geometry pass flagged edges of cell c (bit j-1 = the edge ending at row entry j, j = n
// being the closing edge) as possibly short.  Each edge is seen by its two cells in opposite
// directions: it is reported from the cell that traverses it from the smaller to the larger
// (current) vertex index.
__device__ __forceinline__ void t1_report_cell(const Dev& d, const Consts& k, int c, int n, unsigned smask, unsigned parity) {
  while (smask) {
    const int j = __ffs(smask);     // edge (j-1) -> (j mod n)
    smask &= smask - 1u;
    const int va = row_entry(d.cv, k.N, c, j - 1), vb = row_entry(d.cv, k.N, c, j == n ? 0 : j);
    if (va < vb) t1_mark_edge(d, k, va, vb, parity, kMarkFirstPass);
  }
}

// ---------------------------------------------------------------------------------------------
// rows a4 + a1 + a5: director update (R8, R16), geometry of the moved tiling
// (R14) and short-edge detection (R9).
// d.pos is the position buffer AFTER the move.  kStep = false gives the plain geometry refresh
// used at creation / after avm_set_positions (no noise, no detection).
//
// One thread per cell.  Row entries 0..7 come from planes 0 and 1 (two coalesced 128-bit loads);
// their positions are gathered with up to eight independent predicated 128-bit loads, and the
// director arithmetic (Philox, Box-Muller, sincos) is placed between issuing those gathers and
// consuming them.  Entries beyond the cell's n are copies of entry 0 (r = 0): the edge into the
// first of them is the closing edge and the rest are exact no-ops, so the eight-entry head has a
// fixed trip count and no divergent exits.  Only lanes whose cell has more than 8 vertices (4 %
// of a Voronoi tiling) run the tail over planes 2.. .
// Cells are walked in DESCENDING index order while force_move walks vertices in ascending order,
// so each pass starts on the lines the previous pass touched last (L2 recency).
// ---------------------------------------------------------------------------------------------
// kCoh: every load of data another CTA may have written earlier in the same launch goes through
// the coherent path (the persistent multi-step kernel); false = the per-step kernel, where the
// streams are read with cache hints and the gathers through the non-coherent path.
// kCoh = 2 (the persistent kernel as ONE CTA): everything was written by this very SM, whose L1 is write-through
// and coherent with its own stores, so plain cached loads are safe and a round trip costs an L1 hit instead of L2.
template <int kCoh, typename T> __device__ __forceinline__ T cu_stream(const T* p) { return kCoh == 1 ? __ldcg(p) : kCoh == 2 ? *p : ld_stream(p); }
template <int kCoh> __device__ __forceinline__ double2 cu_pos(const pos_t* p, const Consts& k) {
  return kCoh == 1 ? pos_ldcg(p, k) : kCoh == 2 ? pos_ld(p, k) : pos_ldg(p, k);
}
// Observables (NEXT-2; slots documented at observables_partial_kernel below).  kObs: the pass also reduces
// them over the moved tiling it is computing anyway (avm_step_observe): per-thread values, a fixed
// tree over the CTA in shared memory, one partial per CTA and slot; observables_final_kernel finishes.
static constexpr int kObs = 9;
__device__ __forceinline__ double obs_combine(int slot, double a, double b) {
  return slot == 6 ? fmin(a, b) : slot == 7 ? fmax(a, b) : a + b;
}
template <bool kStep, bool kPerCell, int kCoh, bool kObserve = false>
__device__ __forceinline__ void cell_update_body(const Dev& d, const Consts& k, const unsigned long long step, const unsigned parity,
                                                 const int gid, double* __restrict__ obs_partial = nullptr) {
  if (kStep && gid == 0) { d.ctr->flip_done = 0; d.ctr->next_cand = 0; }   // the previous list is long done
  // the bitmap the force/move launch of this step swept with is spent: clear it for the next step's cell pass
  if (kStep && k.clear_dirty && gid < k.nw) d.dirty[(size_t)(parity ^ 1u) * (size_t)k.nw + gid] = 0u;
  const bool valid = gid < k.N;
  const int c = valid ? k.N - 1 - gid : 0;
  const pos_t* __restrict__ pos = d.pos;
  const int n = valid ? cu_stream<kCoh>(d.cvn + c) : 0;
  const int4 qa = cu_stream<kCoh>(d.cv + c), qb = cu_stream<kCoh>(d.cv + k.N + c);
  const int e[8] = {qa.x, qa.y, qa.z, qa.w, qb.x, qb.y, qb.z, qb.w};
  double th = cu_stream<kCoh>(d.theta + c);
  const unsigned int tag = (unsigned int)cu_stream<kCoh>(d.ctag + c);
  double2 h[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) h[j] = cu_pos<kCoh>(pos + e[j], k);   // padding entries repeat entry 0: r = 0, no predicate
  // ---- director (independent of the gathers above) ----
  if (kStep) {
    th += k.amp * director_noise(k, step, (unsigned long long)tag);
    if (valid) d.theta[c] = th;
  }
  double sn, cs;
  sincos_any(th, &sn, &cs);
  // ---- unwrap relative to entry 0 (R14); |r| >= L/2 is decided conservatively on the high
  // words with integer ALU operations, the exact minimum image runs only where that fires ----
  const unsigned hmin = min(hi_word(k.hLx), hi_word(k.hLy)), hlc = hi_word(k.lc2);
  double rx[8], ry[8];
  unsigned far = 0;
#pragma unroll
  for (int j = 1; j < 8; ++j) {
    rx[j] = __dsub_rn(h[j].x, h[0].x);
    ry[j] = __dsub_rn(h[j].y, h[0].y);
    far = max(far, max(hi_word(rx[j]) & 0x7fffffffu, hi_word(ry[j]) & 0x7fffffffu));
  }
  if (far >= hmin) {
#pragma unroll
    for (int j = 1; j < 8; ++j) { rx[j] = min_image(rx[j], k.Lx, k.hLx); ry[j] = min_image(ry[j], k.Ly, k.hLy); }
  }
  // ---- observing pass: squared unwrapped displacement of the row's vertices since the MSD reference; every
  // vertex belongs to exactly three rows, so the sum over cells is three times the sum over vertices ----
  double msd3 = 0.0;
  if (kObserve) {
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      if (j < n) {
        const int t = d.vtag[e[j]];
        const int2 im = d.img[t];
        const double2 r0 = d.msd_ref[t];
        const double ux = (h[j].x + (double)im.x * k.Lx) - r0.x, uy = (h[j].y + (double)im.y * k.Ly) - r0.y;
        msd3 += ux * ux + uy * uy;
      }
    }
  }
  // ---- shoelace + perimeter; bit j-1 of smask = the edge ending at row entry j looks short ----
  double acc = 0.0, per = 0.0, rxp = 0.0, ryp = 0.0;
  unsigned smask = 0;
#pragma unroll
  for (int j = 1; j < 8; ++j) {
    const double l2 = geom_edge(rxp, ryp, rx[j], ry[j], acc, per);
    if (kStep && hi_word(l2) <= hlc) smask |= 1u << (j - 1);
    rxp = rx[j]; ryp = ry[j];
  }
  // ---- entries 8.. (planes 2..): divergent, only the lanes that hold such a cell ----
  if (n > 8) {
    for (int q = 2; 4 * q < n; ++q) {
      const int j0 = 4 * q;
      const int4 qq = kCoh == 1 ? __ldcg(d.cv + (size_t)q * k.N + c) : d.cv[(size_t)q * k.N + c];
      const int ee[4] = {qq.x, qq.y, qq.z, qq.w};
      double2 hh[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        hh[i] = h[0];
        if (j0 + i < n) hh[i] = cu_pos<kCoh>(pos + ee[i], k);
      }
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        if (j0 + i < n) {
          const double x = min_image(__dsub_rn(hh[i].x, h[0].x), k.Lx, k.hLx);
          const double y = min_image(__dsub_rn(hh[i].y, h[0].y), k.Ly, k.hLy);
          const double l2 = geom_edge(rxp, ryp, x, y, acc, per);
          if (kStep && hi_word(l2) <= hlc) smask |= 1u << (j0 + i - 1);
          rxp = x; ryp = y;
          if (kObserve) {
            const int t = d.vtag[ee[i]];
            const int2 im = d.img[t];
            const double2 r0 = d.msd_ref[t];
            const double ux = (hh[i].x + (double)im.x * k.Lx) - r0.x, uy = (hh[i].y + (double)im.y * k.Ly) - r0.y;
            msd3 += ux * ux + uy * uy;
          }
        }
      }
    }
  }
  {  // closing edge of an n >= 8 cell (an exact no-op for smaller ones, which closed above)
    const double l2 = geom_edge(rxp, ryp, 0.0, 0.0, acc, per);
    if (kStep && hi_word(l2) <= hlc) smask |= 1u << ((n > 8 ? n : 8) - 1);
  }
  if (kObserve) {
    // slots as in observables_partial_kernel; threads beyond the last cell contribute the identities
    __shared__ double sm[kObs][kCellBlock];
    const double A = __dmul_rn(0.5, acc), P = per;
    double x[kObs] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 1.0e300, -1.0e300, 0.0};
    if (valid) {
      const CellPar q = cell_params(d, k, c);
      x[0] = q.KA * (A - q.A0) * (A - q.A0) + q.KP * (P - q.P0) * (P - q.P0);
      x[1] = A; x[2] = P;
      if (A > 0.0) x[3] = P / sqrt(A); else x[4] = 1.0;
      x[5] = A * A; x[6] = A; x[7] = A; x[8] = msd3;
    }
#pragma unroll
    for (int q = 0; q < kObs; ++q) sm[q][threadIdx.x] = x[q];
    __syncthreads();
    for (int st = kCellBlock / 2; st > 0; st >>= 1) {
      if ((int)threadIdx.x < st)
#pragma unroll
        for (int q = 0; q < kObs; ++q) sm[q][threadIdx.x] = obs_combine(q, sm[q][threadIdx.x], sm[q][threadIdx.x + st]);
      __syncthreads();
    }
    if (threadIdx.x < kObs) obs_partial[(size_t)threadIdx.x * gridDim.x + blockIdx.x] = sm[threadIdx.x][0];
  }
  if (!valid) return;
  CellRec r;
  if (kPerCell) rec_from_geometry(d.par[c], __dmul_rn(0.5, acc), per, r.a, r.p);   // Eq. 1 per cell (NEXT-4); written by no kernel
  else { r.a = k.KA2 * (__dmul_rn(0.5, acc) - k.A0); r.p = k.KP2 * (per - k.P0); }   // Eq. A1
  r.nx = cs; r.ny = sn;
  st_rec(d.rec + c, r);
  smask &= n >= 32 ? ~0u : (1u << n) - 1u;     // edges beyond the closing one are padding
  if (kStep && smask) t1_report_cell(d, k, c, n, smask, parity);
}
// the observing instantiation of the per-step pass (the last step of avm_step_observe)
template <bool kPerCell>
__global__ void __launch_bounds__(kCellBlock)
cell_update_observe_kernel(const __grid_constant__ Dev d, const __grid_constant__ Consts k, const unsigned long long step,
                           const unsigned parity, double* __restrict__ obs_partial) {
  pdl_launch_dependents();
  pdl_wait();
  cell_update_body<true, kPerCell, 0, true>(d, k, step, parity, blockIdx.x * kCellBlock + threadIdx.x, obs_partial);
}
template <bool kStep, bool kPerCell>
__global__ void __launch_bounds__(kCellBlock, AVM_CU_MINB)
cell_update_kernel(const __grid_constant__ Dev d, const __grid_constant__ Consts k, const unsigned long long step,
                   const unsigned parity) {
  pdl_launch_dependents();
  pdl_wait();
  cell_update_body<kStep, kPerCell, 0>(d, k, step, parity, blockIdx.x * kCellBlock + threadIdx.x);
}

// Detection alone (test hooks avm_t1_pass / avm_debug_t1): thread per vertex, edge owned by the
// smaller current index.
__global__ void detect_mark_kernel(const __grid_constant__ Dev d, const __grid_constant__ Consts k, const unsigned parity,
                                   const bool count_stats) {
  const int v = blockIdx.x * blockDim.x + threadIdx.x;
  if (v >= k.V) return;
  const double2 h = pos_ld(d.pos + v, k);
  for (int s = 0; s < 3; ++s) {
    const int w = d.vn[s * k.Vs + v];
    if (v < w) {
      // cheap pre-test; t1_mark_edge repeats the canonical one
      const double2 q = pos_ld(d.pos + w, k);
      const double dx = min_image(q.x - h.x, k.Lx, k.hLx), dy = min_image(q.y - h.y, k.Ly, k.hLy);
      if (dx * dx + dy * dy < k.lc2) t1_mark_edge(d, k, v, w, parity, count_stats ? kMarkFirstPass : kMarkSilent);
    }
  }
}

// Repeated passes (NEXT-1; "called repeatedly until no changes").  A further pass
// on the current state can only find candidates among the edges that have an endpoint in a cell
// of a candidate of the previous pass: lengths changed only at flipped vertices, eligibility
// (R10) only through the vertex counts of a flipped candidate's four cells, and blocked
// candidates are such edges themselves.  So one more pass =
//   release : clear the minimum keys of the previous pass's list, empty the new list;
//   detect  : one warp per previous candidate tests the edges of every vertex of its four cells
//             (each edge once per pass: stamp on the half-edge of its smaller endpoint) and marks;
//   flip    : t1_flip_kernel on the new list.
// When a pass found nothing, the following ones have nothing to release, test or flip.
__global__ void __launch_bounds__(kT1Block)
t1_release_kernel(const __grid_constant__ Dev d, const __grid_constant__ Consts k, const unsigned list, const int empty_list) {
  pdl_launch_dependents();
  pdl_wait();
  const unsigned n = min(d.ctr->n_cand[list], list_cap(k, list));
  const Cand* __restrict__ l = list_base(d, k, list);
  for (unsigned int i = blockIdx.x * kT1Block + threadIdx.x; i < n; i += gridDim.x * kT1Block) {
    const Cand c = l[i];
    d.minkey[c.cL] = ~0ull; d.minkey[c.cR] = ~0ull; d.minkey[c.cE1] = ~0ull; d.minkey[c.cE2] = ~0ull;
  }
  if (empty_list >= 0 && blockIdx.x == 0 && threadIdx.x == 0) d.ctr->n_cand[empty_list] = 0;
}

__global__ void __launch_bounds__(kT1Block)
t1_local_detect_kernel(const __grid_constant__ Dev d, const __grid_constant__ Consts k, const unsigned list_prev,
                       const unsigned list_new, const unsigned stamp) {
  pdl_launch_dependents();
  pdl_wait();
  const unsigned n = min(d.ctr->n_cand[list_prev], list_cap(k, list_prev));
  const Cand* __restrict__ l = list_base(d, k, list_prev);
  const int lane = threadIdx.x & 31;
  const unsigned gwarp = (blockIdx.x * kT1Block + threadIdx.x) >> 5, nwarps = (gridDim.x * kT1Block) >> 5;
  for (unsigned int i = gwarp; i < n; i += nwarps) {
    const Cand c = l[i];
    const int quad[4] = {c.cL, c.cR, c.cE1, c.cE2};
#pragma unroll 1
    for (int t = 0; t < 4; ++t) {
      const int nrow = d.cvn[quad[t]];
      if (lane >= nrow) continue;
      const int u = row_entry(d.cv, k.N, quad[t], lane);
      const double2 hu = pos_ld(d.pos + u, k);
#pragma unroll 1
      for (int sl = 0; sl < 3; ++sl) {
        const int wv = d.vn[sl * k.Vs + u];
        // the half-edge of the smaller endpoint identifies the edge
        int owner = u, other = wv, oslot = sl;
        if (wv < u) {
          owner = wv; other = u;
          oslot = d.vn[wv] == u ? 0 : d.vn[k.Vs + wv] == u ? 1 : 2;
        }
        if (atomicExch(&d.estamp[(size_t)oslot * k.Vs + owner], stamp) == stamp) continue;   // tested in this pass already
        const double2 hw = pos_ld(d.pos + wv, k);
        const double dx = min_image(hw.x - hu.x, k.Lx, k.hLx), dy = min_image(hw.y - hu.y, k.Ly, k.hLy);
        if (dx * dx + dy * dy < k.lc2) t1_mark_edge(d, k, owner, other, list_new, kMarkRepeatedPass);
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// rows a6 (deciding half) + a7: flip + rewrite (R9 geometry, R12 lists).  FOUR LANES per candidate:
// lane t of a group owns cell t of the candidate's quadruple (L, R, E1, E2), so a warp carries
// eight candidates at once.  A candidate flips iff its key is the minimum recorded on all four of
// its cells (R11); winners therefore own disjoint cell quadruples and every word written below
// belongs to a vertex or row inside the winner's own quadruple.  minkey is only read here.
// Handles candidates base .. base+7 (< n) of `list`; returns how many of them flipped (warp-uniform).
// Used by the stand-alone T1 kernel and by the flippers of the fused force_move launch.
// ---------------------------------------------------------------------------------------------
// kR = number of row entries held per lane: 16 (rows live in registers, every index is static and
// all loads of a phase are in flight together) for S <= 16, 32 (a local array) for larger strides.
template <int kR> using RowIdx = std::make_integer_sequence<int, kR>;
// position of `mark` among the first n entries (rows hold distinct vertices; 0 if absent)
template <int kR, int... J>
__device__ __forceinline__ int row_find(const int (&r)[kR], const int n, const int mark, std::integer_sequence<int, J...>) {
  int p = 0;
  ((p = (J < n && r[J] == mark) ? J : p), ...);
  return p;
}
// w = r without entry p (later entries shift down)
template <int kR, int... J>
__device__ __forceinline__ void row_delete(const int (&r)[kR], int (&w)[kR], const int p, std::integer_sequence<int, J...>) {
  ((w[J] = J < p ? r[J] : r[J + 1 < kR ? J + 1 : kR - 1]), ...);
}
// w = r with `ins` inserted immediately after entry p (later entries shift up)
template <int kR, int... J>
__device__ __forceinline__ void row_insert(const int (&r)[kR], int (&w)[kR], const int p, const int ins, std::integer_sequence<int, J...>) {
  ((w[J] = J <= p ? r[J] : J == p + 1 ? ins : r[J > 0 ? J - 1 : 0]), ...);
}
// r = w with the entries from n on replaced by entry 0
template <int kR, int... J>
__device__ __forceinline__ void row_pad(const int (&w)[kR], int (&r)[kR], const int n, std::integer_sequence<int, J...>) {
  ((r[J] = J < n ? w[J] : w[0]), ...);
}
template <int kR>
__device__ __forceinline__ unsigned t1_flip_quads_impl(const Dev& d, const Consts& k, const Cand* __restrict__ list,
                                                       const unsigned base, const unsigned n, const int lane_in,
                                                       const int4* __restrict__ pre) {
  // pre (optional): the 64 bytes of this lane's candidate, fetched by the caller before the list length was known
  const int lane = lane_in & 31;
  const int t = lane & 3;
  const unsigned i = base + (unsigned)(lane >> 2);
  const bool have = i < n;
  // ---- everything is read before anything is written; the loads of a phase are independent of
  // one another (the marking thread decoded the neighbourhood), so the decision costs no extra
  // round trip: phase 1 = the candidate, phase 2 = keys, rows and the two end points
  int4 ca = make_int4(0, 0, 0, 0), cb = ca, cc = ca, cd = ca;
  if (pre) {
    if (have) { ca = pre[0]; cb = pre[1]; cc = pre[2]; cd = pre[3]; }
  } else if (have) {
    const int4* __restrict__ src = reinterpret_cast<const int4*>(list + i);
    ca = __ldcg(src); cb = __ldcg(src + 1); cc = __ldcg(src + 2); cd = __ldcg(src + 3);
  }
  const int v1 = ca.x, v2 = ca.y, k1 = ca.z, k2 = ca.w;
  const int cL = cb.x, cR = cb.y, cE1 = cb.z, cE2 = cb.w;
  const unsigned long long key = ((unsigned long long)(unsigned)cc.y << 32) | (unsigned)cc.x;
  const int sx1 = cc.z & 3, sx2 = (cc.z >> 2) & 3;
  const int x1 = cd.x, y1 = cd.y, x2 = cd.z, y2 = cd.w;
  const int cell = t == 0 ? cL : t == 1 ? cR : t == 2 ? cE1 : cE2;     // 0 for idle groups: a valid index
  const unsigned long long mk = __ldcg(d.minkey + cell);      // written by L2 atomics: never from L1
  const int nrow = (cc.w >> (8 * t)) & 0xff;            // as counted by the marking thread (a winner's cells are its own)
  const int need = t < 2 ? nrow : nrow + 1;             // entries of the longer of the old and the new row
  const double2 h1 = pos_ld(d.pos + v1, k), h2 = pos_ld(d.pos + v2, k);
  // planes 0 and 1 always (their padding is part of the cell pass's fixed-trip head), later planes only when the
  // row reaches them: nobody reads the padding of a plane the row does not reach
  int r[kR];
#pragma unroll
  for (int q = 0; q < kR / 4; ++q) {
    int4 e = make_int4(0, 0, 0, 0);
    if (4 * q < k.S && (q < 2 || 4 * q < need)) e = d.cv[(size_t)q * k.N + cell];
    r[4 * q] = e.x; r[4 * q + 1] = e.y; r[4 * q + 2] = e.z; r[4 * q + 3] = e.w;
  }
  const unsigned agree = __ballot_sync(kFull, have && mk == key);
  const unsigned wins = __ballot_sync(kFull, ((agree >> (lane & ~3)) & 0xfu) == 0xfu);
  const unsigned nflips = (unsigned)__popc(wins & 0x11111111u);
  if (!((wins >> lane) & 1u)) return nflips;
  // ---- geometry: rigid counter-clockwise quarter turn about the midpoint, new length 1.5 l_c (R9);
  // every lane of the group evaluates it (same bits) because each needs both new positions below
  const double dx = min_image(h2.x - h1.x, k.Lx, k.hLx), dy = min_image(h2.y - h1.y, k.Ly, k.hLy);
  const double l = sqrt(dx * dx + dy * dy);
  const double mx = h1.x + 0.5 * dx, my = h1.y + 0.5 * dy;
  double px = 0.0, py = 1.0;
  if (l > 0.0) { px = -dy / l; py = dx / l; }
  const double half = 0.75 * k.lc;
  // (pos_round: the value the stored position reads back as; the identity in the fp64 build)
  const double2 n2 = pos_round(make_double2(wrap_box(mx + half * px, k.Lx), wrap_box(my + half * py, k.Ly)), k);
  const double2 n1 = pos_round(make_double2(wrap_box(mx - half * px, k.Lx), wrap_box(my - half * py, k.Ly)), k);
  // ---- lists: u = ([w, x, y]; [C0, C1, C2]) cyclic from the partner slot
  //          -> ([w, y, z]; [C1, C2, C']), z = partner's old x, C' = partner's old C1 (R12);
  // outer vertices: x1 was joined to v1 and is now joined to v2 (same slot), x2 likewise.
  // Lane 0 rewrites v1, lane 1 v2, lane 2 x1, lane 3 x2.
  if (t < 2) {
    // unwrapped positions (MSD): the end point moved from h to (m -+ half p) before wrapping; count the box lengths
    const double ux = t == 0 ? mx - half * px : h2.x - 0.5 * dx + half * px, uy = t == 0 ? my - half * py : h2.y - 0.5 * dy + half * py;
    const double2 nn = t == 0 ? n1 : n2;
    const int ix = __double2int_rn((ux - nn.x) / k.Lx), iy = __double2int_rn((uy - nn.y) / k.Ly);
    if (ix | iy) {
      int2* im = d.img + d.vtag[t == 0 ? v1 : v2];
      int2 c = *im; c.x += ix; c.y += iy; *im = c;     // unwrapped = wrapped + count x L
    }
  }
  if (t == 0) {
    const int a1 = (k1 + 1) % 3, b1 = (k1 + 2) % 3;
    pos_st(d.pos + v1, n1, k);
    d.vn[a1 * k.Vs + v1] = y1; d.vn[b1 * k.Vs + v1] = x2;
    d.vc[k1 * k.Vs + v1] = cE1; d.vc[a1 * k.Vs + v1] = cR; d.vc[b1 * k.Vs + v1] = cE2;
  } else if (t == 1) {
    const int a2 = (k2 + 1) % 3, b2 = (k2 + 2) % 3;
    pos_st(d.pos + v2, n2, k);
    d.vn[a2 * k.Vs + v2] = y2; d.vn[b2 * k.Vs + v2] = x1;
    d.vc[k2 * k.Vs + v2] = cE2; d.vc[a2 * k.Vs + v2] = cL; d.vc[b2 * k.Vs + v2] = cE1;
  } else if (t == 2) {
    d.vn[sx1 * k.Vs + x1] = v2;
  } else {
    d.vn[sx2 * k.Vs + x2] = v1;
  }
  __syncwarp(wins);     // reconverge: the four lanes of a group must issue the loads below together
  // ---- my row: L deletes v1, R deletes v2 (later entries shift down); E1 inserts v2 immediately
  // after v1, E2 inserts v1 immediately after v2 (later entries shift up); padding repeats entry 0.
  // All indices are static so that the row stays in registers.
  const int mark = (t & 1) ? v2 : v1;             // L, E1 look for v1; R, E2 look for v2
  const int ins = t == 2 ? v2 : v1;
  // (fold expressions over the entry index instead of loops: every index is a literal, so the row
  // is scalarised into registers whatever the optimiser makes of the conditions)
  const int p = row_find(r, nrow, mark, RowIdx<kR>{});
  int w[kR];
  int nnew;
  if (t < 2) { row_delete(r, w, p, RowIdx<kR>{}); nnew = nrow - 1; }
  else { row_insert(r, w, p, ins, RowIdx<kR>{}); nnew = nrow + 1; }      // nrow < S (R10): nothing falls off
  __syncwarp(wins);
  row_pad(w, r, nnew, RowIdx<kR>{});                                      // r = the new row, padding repeats entry 0
  const int e0 = r[0];
#pragma unroll
  for (int q = 0; q < kR / 4; ++q)
    if (4 * q < k.S && (q < 2 || 4 * q < need)) d.cv[(size_t)q * k.N + cell] = make_int4(r[4 * q], r[4 * q + 1], r[4 * q + 2], r[4 * q + 3]);
  d.cvn[cell] = nnew;
  // ---- refresh the cached geometry of my cell (directors unchanged): the same serial sum as the
  // per-step pass (geom_edge), so that a resumed run reproduces these records bit for bit.  Positions
  // are fetched eight at a time with unconditional, mutually independent loads (entries beyond the
  // row repeat entry 0: a valid index, the same sector); v1 and v2 take their new positions from
  // registers whatever the loads return.
  const double2 g0 = pos_ld(d.pos + e0, k);
  const double2 h0 = e0 == v1 ? n1 : e0 == v2 ? n2 : g0;
  double rxp = 0.0, ryp = 0.0, acc = 0.0, per = 0.0;
#pragma unroll
  for (int b = 0; 1 + 8 * b < kR; ++b) {
    if (1 + 8 * b < nnew) {
      double2 g[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        g[u] = g0;
        if (1 + 8 * b + u < kR) g[u] = pos_ld(d.pos + r[1 + 8 * b + u < kR ? 1 + 8 * b + u : 0], k);
      }
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        if (1 + 8 * b + u < kR && 1 + 8 * b + u < nnew) {
          const int e = r[1 + 8 * b + u < kR ? 1 + 8 * b + u : 0];
          const double2 hu = e == v1 ? n1 : e == v2 ? n2 : g[u];
          const double rx = min_image(__dsub_rn(hu.x, h0.x), k.Lx, k.hLx);
          const double ry = min_image(__dsub_rn(hu.y, h0.y), k.Ly, k.hLy);
          geom_edge(rxp, ryp, rx, ry, acc, per);
          rxp = rx; ryp = ry;
        }
      }
    }
  }
  geom_edge(rxp, ryp, 0.0, 0.0, acc, per);      // the closing edge back to entry 0
  double ra, rp;
  if (k.per_cell) rec_from_geometry(d.par[cell], __dmul_rn(0.5, acc), per, ra, rp);
  else { ra = k.KA2 * (__dmul_rn(0.5, acc) - k.A0); rp = k.KP2 * (per - k.P0); }
  rec_st_ap(d.rec + cell, ra, rp);
  return nflips;
}
__device__ __noinline__ unsigned t1_flip_quads(const Dev& d, const Consts& k, const Cand* __restrict__ list, const unsigned base,
                                               const unsigned n, const int lane) {
  return k.S <= 16 ? t1_flip_quads_impl<16>(d, k, list, base, n, lane) : t1_flip_quads_impl<32>(d, k, list, base, n, lane);
}

__global__ void __launch_bounds__(kT1Block)
t1_flip_kernel(const __grid_constant__ Dev d, const __grid_constant__ Consts k, const unsigned parity, const bool count_stats) {
  pdl_launch_dependents();
  pdl_wait();
  const Cand* __restrict__ list = list_base(d, k, parity);
  const int lane = threadIdx.x & 31;
  const unsigned gwarp = (blockIdx.x * kT1Block + threadIdx.x) >> 5, nwarps = (gridDim.x * kT1Block) >> 5;
  // the first batch of candidate records is fetched while the list length is still in flight (one round trip
  // less in a kernel that is a chain of round trips); entries beyond the length are ignored
  int4 pre[4] = {make_int4(0, 0, 0, 0), make_int4(0, 0, 0, 0), make_int4(0, 0, 0, 0), make_int4(0, 0, 0, 0)};
  {
    const unsigned i0 = gwarp * 8u + (unsigned)(lane >> 2);
    if (i0 < list_cap(k, parity)) {
      const int4* __restrict__ src = reinterpret_cast<const int4*>(list + i0);
      pre[0] = __ldcg(src); pre[1] = __ldcg(src + 1); pre[2] = __ldcg(src + 2); pre[3] = __ldcg(src + 3);
    }
  }
  const unsigned int n_cand = min(__ldcg(&d.ctr->n_cand[parity]), list_cap(k, parity));
  if (count_stats && gwarp == 0 && lane == 0 && n_cand) atomicAdd((unsigned long long*)&d.ctr->t1_candidates, (unsigned long long)n_cand);
  if (count_stats && parity < 2u && gwarp == 0 && lane == 0) report_t1_load(d, n_cand);     // the step's list: report the T1 load
  unsigned int flips = 0, seen = 0;
  // the implementation is inlined here (pointers and constants come straight from the kernel's
  // constant bank; the row stays in registers): the kernel is a chain of dependent round trips and
  // every reload or local-memory access in it would queue behind the outstanding gathers
  for (unsigned int i = gwarp * 8u; i < n_cand; i += nwarps * 8u) {
    flips += k.S <= 16 ? t1_flip_quads_impl<16>(d, k, list, i, n_cand, lane, i == gwarp * 8u ? pre : nullptr)
                       : t1_flip_quads(d, k, list, i, n_cand, lane);
    seen += min(8u, n_cand - i);
  }
  if (count_stats && lane == 0) {
    if (flips) atomicAdd((unsigned long long*)&d.ctr->t1_flips, (unsigned long long)flips);
    if (seen - flips) atomicAdd((unsigned long long*)&d.ctr->t1_blocked, (unsigned long long)(seen - flips));
  }
}

// ---------------------------------------------------------------------------------------------
// Launch-free stepping ("entirely on the GPU"): ONE cooperative
// launch advances n_steps timesteps.  The three stages of a step (rows a2+a3; a4+a1+a5+a6; a6+a7) are
// the same device functions as in the per-step kernels, separated by grid-wide barriers instead of
// kernel boundaries; loads of data written earlier in the launch take the coherent path.  Used
// for systems that fit in L2 and are bound by launch latency, not bandwidth (configs 0-2); the
// results are bit-identical to the per-step schedules.  A grid of one CTA needs no barrier but
// __syncthreads (grid.sync() of a one-CTA cooperative grid is just that).
// ---------------------------------------------------------------------------------------------
// Grid-wide barrier of the cooperative launch (every CTA is resident).  Monotonic arrival counter, zeroed by
// the host before the launch; `epoch` counts the barriers passed.  Release: fence, then arrive; acquire: observe
// the full count, then fence.  One CTA: __syncthreads is all it takes.
struct GridBarrier {
  unsigned int* bar;
  unsigned int epoch;
  bool cluster;     // the whole grid is ONE thread-block cluster: the hardware cluster barrier (release / acquire at cluster scope)
  __device__ __forceinline__ void sync() {
    ++epoch;
    if (gridDim.x == 1) { __syncthreads(); return; }
    if (cluster) {
      asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
      return;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
      __threadfence();
      atomicAdd(bar, 1u);
      const unsigned target = epoch * gridDim.x;
      while (ld_volatile(bar) < target) { }
      __threadfence();
    }
    __syncthreads();
  }
};
// CTA size of the persistent kernel in all its forms (one CTA, one cluster, cooperative grid): its launch bounds, the
// occupancy query that sizes the cooperative grid and both launches use this one constant, whatever AVM_VERTEX_BLOCK
// is.  Measured at configs[1] as one cluster: 256 threads 7.7 us/step, 512 threads 8.4.
static constexpr int kClusterBlock = 256;
template <bool kPerCell, bool kOneCta>
__global__ void __launch_bounds__(kClusterBlock)
persistent_steps_kernel(Dev d, const __grid_constant__ Consts k, const unsigned long long step0, const int n_steps, const int one_cluster) {
  GridBarrier grid = {&d.ctr->bar, 0u, one_cluster != 0};
  const int tid = blockIdx.x * blockDim.x + threadIdx.x, stride = gridDim.x * blockDim.x;
  const int lane = threadIdx.x & 31;
  const unsigned gwarp = (unsigned)tid >> 5, nwarps = (unsigned)stride >> 5;
  const int n_round = (k.N + 31) & ~31;                 // the cell body wants whole warps (it uses no warp collectives, but stays uniform)
  for (int it = 0; it < n_steps; ++it) {
    const unsigned long long step = step0 + (unsigned long long)it;
    const unsigned parity = (unsigned)(step & 1ull);
    // ---- rows a2 + a3 (and the release of the previous step's minimum keys, row a6)
    const unsigned prev = min(__ldcg(&d.ctr->n_cand[parity ^ 1u]), (unsigned)k.cap_a);
    if (tid == 0) d.ctr->n_cand[parity] = 0;           // this step's list; its previous contents were last read two stages ago
    for (unsigned i = tid; i < prev; i += stride) {
      const int4 q = __ldcg(reinterpret_cast<const int4*>(d.cand + i) + 1);
      d.minkey[q.x] = ~0ull; d.minkey[q.y] = ~0ull; d.minkey[q.z] = ~0ull; d.minkey[q.w] = ~0ull;
    }
    if (kOneCta) {
      for (int v = tid; v < k.V; v += stride) move_vertex_plain(d, k, v);
    } else {
      // two vertices per trip: both sets of loads are in flight together (a cluster takes 2 vertices per thread at 8192)
      int v = tid;
      for (; v + stride < k.V; v += 2 * stride) move_two_coherent(d, k, v, v + stride);
      if (v < k.V) move_vertex_coherent(d, k, v);
    }
    grid.sync();
    { pos_t* t = d.pos; d.pos = d.pos_next; d.pos_next = t; }
    // ---- rows a4 + a1 + a5 + a6 (marking half)
    for (int gid = tid; gid < n_round; gid += stride) cell_update_body<true, kPerCell, kOneCta ? 2 : 1>(d, k, step, parity, gid);
    grid.sync();
    // ---- rows a6 (deciding half) + a7
    const unsigned n_cand = min(__ldcg(&d.ctr->n_cand[parity]), (unsigned)k.cap_a);
    if (n_cand) {                                        // uniform over the grid: read after the barrier
      if (tid == 0) atomicAdd((unsigned long long*)&d.ctr->t1_candidates, (unsigned long long)n_cand);
      unsigned flips = 0, seen = 0;
      for (unsigned i = gwarp * 8u; i < n_cand; i += nwarps * 8u) {
#if AVM_PERS_FLIP_INLINE
        flips += k.S <= 16 ? t1_flip_quads_impl<16>(d, k, d.cand, i, n_cand, lane) : t1_flip_quads(d, k, d.cand, i, n_cand, lane);
#else
        flips += t1_flip_quads(d, k, d.cand, i, n_cand, lane);
#endif
        seen += min(8u, n_cand - i);
      }
      if (lane == 0) {
        if (flips) atomicAdd((unsigned long long*)&d.ctr->t1_flips, (unsigned long long)flips);
        if (seen - flips) atomicAdd((unsigned long long*)&d.ctr->t1_blocked, (unsigned long long)(seen - flips));
      }
      grid.sync();
    }
  }
}

// Clears the minimum keys of both candidate lists and empties them (before a re-sort, around the
// test hooks).  Inside avm_step this work rides in force_move's prologue instead.
__global__ void __launch_bounds__(kT1Block)
t1_reset_kernel(const Dev d, const unsigned cap) {
  const unsigned n0 = d.ctr->n_cand[0], n1 = d.ctr->n_cand[1];
  const unsigned n = min(n0 > n1 ? n0 : n1, cap);
  for (unsigned int i = blockIdx.x * kT1Block + threadIdx.x; i < n; i += gridDim.x * kT1Block) {
    const Cand c = d.cand[i];
    d.minkey[c.cL] = ~0ull; d.minkey[c.cR] = ~0ull; d.minkey[c.cE1] = ~0ull; d.minkey[c.cE2] = ~0ull;
  }
}
__global__ void zero_counts_kernel(const Dev d) { d.ctr->n_cand[0] = 0; d.ctr->n_cand[1] = 0; d.ctr->n_cand[2] = 0; d.ctr->n_cand[3] = 0; d.ctr->n_win = 0; d.ctr->flip_done = 0; d.ctr->next_cand = 0; }

// debug hook: winners without flipping; (tag_min, tag_max) pairs out
__global__ void t1_debug_kernel(const Dev d, int* cand_pairs, int* win_pairs, long long capacity) {
  const unsigned int n_cand = d.ctr->n_cand[0];
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
  cell_area_perimeter(d.pos, d.cv, c, d.cvn[c], k, A, P);
  ap[c] = make_double2(A, P);
  if (ap_user) {
    const int t = d.ctag[c];
    ap_user[2 * t] = A; ap_user[2 * t + 1] = P;
  }
}

__global__ void forces_kernel(const Dev d, const Consts k, const double2* __restrict__ ap, double* __restrict__ force_user) {
  const int v = blockIdx.x * blockDim.x + threadIdx.x;
  if (v >= k.V) return;
  const double2 h = pos_ld(d.pos + v, k);
  CellRec c[3];
  double2 q[3];
#pragma unroll
  for (int s = 0; s < 3; ++s) {
    q[s] = pos_ld(d.pos + d.vn[s * k.Vs + v], k);
    const int cell = d.vc[s * k.Vs + v];
    const double2 a = ap[cell];
    if (k.per_cell) rec_from_geometry(d.par[cell], a.x, a.y, c[s].a, c[s].p);
    else { c[s].a = k.KA2 * (a.x - k.A0); c[s].p = k.KP2 * (a.y - k.P0); }
    c[s].nx = 0.0; c[s].ny = 0.0;
  }
  const double2 f = vertex_force(h, q[0], q[1], q[2], c[0], c[1], c[2], k);
  const int t = d.vtag[v];
  force_user[2 * t] = f.x; force_user[2 * t + 1] = f.y;
}

// Observables of the current state (NEXT-2): energy, Eq. 1 / A1, and the
// per-cell statistics a user of the model measures (shape index P / sqrt(A), area moments).
// Slots: 0 energy, 1 sum A, 2 sum P, 3 sum P/sqrt(A) over cells with A > 0, 4 number of cells with
// A <= 0, 5 sum A^2, 6 min A, 7 max A, 8 sum over vertices of the squared unwrapped displacement since the
// MSD reference.  Block partials in a fixed order, finished by one block (deterministic, no
// floating-point atomics).
__device__ __forceinline__ void obs_block_reduce(double (&x)[kObs], double (*sm)[256]) {
#pragma unroll
  for (int q = 0; q < kObs; ++q) sm[q][threadIdx.x] = x[q];
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if (threadIdx.x < s)
#pragma unroll
      for (int q = 0; q < kObs; ++q) sm[q][threadIdx.x] = obs_combine(q, sm[q][threadIdx.x], sm[q][threadIdx.x + s]);
    __syncthreads();
  }
}
__global__ void __launch_bounds__(256)
observables_partial_kernel(const Dev d, const Consts k, double* __restrict__ partial) {
  __shared__ double sm[kObs][256];
  double x[kObs] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 1.0e300, -1.0e300, 0.0};
  for (int c = blockIdx.x * 256 + threadIdx.x; c < k.N; c += gridDim.x * 256) {
    double A, P;
    cell_area_perimeter(d.pos, d.cv, c, d.cvn[c], k, A, P);
    const CellPar q = cell_params(d, k, c);
    x[0] += q.KA * (A - q.A0) * (A - q.A0) + q.KP * (P - q.P0) * (P - q.P0);
    x[1] += A; x[2] += P;
    if (A > 0.0) x[3] += P / sqrt(A); else x[4] += 1.0;
    x[5] += A * A;
    x[6] = fmin(x[6], A); x[7] = fmax(x[7], A);
  }
  // mean-square displacement: unwrapped position = wrapped position + image count x box length
  for (int v = blockIdx.x * 256 + threadIdx.x; v < k.V; v += gridDim.x * 256) {
    const int t = d.vtag[v];
    const double2 h = pos_ld(d.pos + v, k), r0 = d.msd_ref[t];
    const int2 im = d.img[t];
    const double dx = (h.x + (double)im.x * k.Lx) - r0.x, dy = (h.y + (double)im.y * k.Ly) - r0.y;
    x[8] += dx * dx + dy * dy;
  }
  obs_block_reduce(x, sm);
  if (threadIdx.x < kObs) partial[(size_t)threadIdx.x * gridDim.x + blockIdx.x] = sm[threadIdx.x][0];
}
__global__ void __launch_bounds__(256)
observables_final_kernel(const Dev d, const double* __restrict__ partial, int n, const double msd_scale) {
  __shared__ double sm[kObs][256];
  double x[kObs] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 1.0e300, -1.0e300, 0.0};
  for (int i = threadIdx.x; i < n; i += 256)
#pragma unroll
    for (int q = 0; q < kObs; ++q) x[q] = obs_combine(q, x[q], partial[(size_t)q * n + i]);
  obs_block_reduce(x, sm);
  // msd_scale: 1 for a sum over vertices, 1/3 for the sum over the rows of all cells (the observing cell pass)
  if (threadIdx.x < kObs) d.ctr->obs[threadIdx.x] = threadIdx.x == 8 ? sm[8][0] * msd_scale : sm[threadIdx.x][0];
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
int cell_pass_grid(int N) { return cdiv(N, kCellBlock); }

// Grid of the persistent force/move kernel: a whole number of CTAs per SM of the current device,
// never more CTAs than there is work.  Called once per simulation (avm_create); the result lives
// in Consts::fm_grid.
int force_move_grid(int V) {
  int a = 0, b = 0, dev = 0, sms = 148;
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&a, force_move_kernel<true>, kVertexBlock, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, force_move_kernel<false>, kVertexBlock, 0);
  int per_sm = a < b ? a : b;
  if (per_sm < 1) per_sm = 1;
  if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const int want = cdiv(V, kVertexBlock);
  const int cap = sms * per_sm;
  return want < cap ? want : cap;
}

// Launch with the programmatic-stream-serialization attribute (see pdl_wait above).
template <typename... KArgs, typename... Args>
static cudaError_t launch_chained(void (*kernel)(KArgs...), int grid, int block, cudaStream_t s, bool pdl, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)block); cfg.dynamicSmemBytes = 0; cfg.stream = s;
  cudaLaunchAttribute attr[1];
  int na = 0;
  if (pdl) { attr[na].id = cudaLaunchAttributeProgrammaticStreamSerialization; attr[na].val.programmaticStreamSerializationAllowed = 1; ++na; }
  cfg.attrs = attr; cfg.numAttrs = (unsigned)na;
  return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// One timestep.  d.pos = positions at the start of the step, d.pos_next = buffer for the moved
// positions (the caller swaps them afterwards).
//   consume_pending: the previous step left its T1 flips pending; they ride in this force/move launch.
//   leave_pending  : this step leaves its own flips pending (two launches) instead of running the
//                    stand-alone T1 kernel (three launches, the step complete on return).
// ev (optional, AVM_K_COUNT+1 events): recorded before/after each kernel by avm_step_profile.
int launch_step(const Dev& d, const Consts& k, unsigned long long step, cudaStream_t s, cudaEvent_t* ev, bool consume_pending,
                bool leave_pending, double* obs_partial) {
  const unsigned parity = (unsigned)(step & 1ull);
  if (ev) cudaEventRecord(ev[0], s);
  const bool pdl = AVM_PDL && ev == nullptr;   // events between the kernels would break the chain anyway
  if (consume_pending) launch_chained(force_move_kernel<true>, k.fm_grid, kVertexBlock, s, pdl, d, k, step);
  else launch_chained(force_move_kernel<false>, k.fm_grid, kVertexBlock, s, pdl, d, k, step);
  if (ev) cudaEventRecord(ev[1], s);
  Dev m = d;                      // from here on the moved positions are "the" positions
  m.pos = d.pos_next; m.pos_next = d.pos;
  Consts kc = k;
  kc.flag_dirty = leave_pending ? 1 : 0;       // the flagged-vertex bitmap is only needed when the flips stay pending
  kc.clear_dirty = consume_pending ? 1 : 0;    // the bitmap this step's force/move launch swept with is spent
  const int cgrid = cdiv(k.N, kCellBlock);
  int n_launched = leave_pending ? 2 : 3;
  if (obs_partial) {
    // the observing pass: same arithmetic, plus the reduction of the observables of the moved tiling (NEXT-2)
    if (k.per_cell) launch_chained(cell_update_observe_kernel<true>, cgrid, kCellBlock, s, pdl, m, kc, step, parity, obs_partial);
    else launch_chained(cell_update_observe_kernel<false>, cgrid, kCellBlock, s, pdl, m, kc, step, parity, obs_partial);
    observables_final_kernel<<<1, 256, 0, s>>>(m, obs_partial, cgrid, 1.0 / 3.0);
    ++n_launched;
  } else if (k.per_cell) launch_chained(cell_update_kernel<true, true>, cgrid, kCellBlock, s, pdl, m, kc, step, parity);
  else launch_chained(cell_update_kernel<true, false>, cgrid, kCellBlock, s, pdl, m, kc, step, parity);
  if (ev) cudaEventRecord(ev[2], s);
  if (!leave_pending) launch_chained(t1_flip_kernel, kT1Grid, kT1Block, s, pdl && !obs_partial, m, k, parity, true);
  if (ev) cudaEventRecord(ev[3], s);
  return n_launched;
}

// number of edges shorter than l_c in the current state -> ctr->n_win (creation: first guess of the T1 load)
__global__ void count_short_edges_kernel(const Dev d, const Consts k) {
  const int v = blockIdx.x * blockDim.x + threadIdx.x;
  if (v >= k.V) return;
  const double2 h = pos_ld(d.pos + v, k);
  int n = 0;
  for (int s = 0; s < 3; ++s) {
    const int w = d.vn[s * k.Vs + v];
    if (v < w) {
      const double2 q = pos_ld(d.pos + w, k);
      const double dx = min_image(q.x - h.x, k.Lx, k.hLx), dy = min_image(q.y - h.y, k.Ly, k.hLy);
      n += dx * dx + dy * dy < k.lc2;
    }
  }
  if (n) atomicAdd(&d.ctr->n_win, (unsigned)n);
}
int launch_count_short_edges(const Dev& d, const Consts& k, cudaStream_t s) {
  count_short_edges_kernel<<<cdiv(k.V, 256), 256, 0, s>>>(d, k);
  return 1;
}

#ifndef AVM_CLUSTER_VERTICES
#define AVM_CLUSTER_VERTICES 8192
#endif
static constexpr int kClusterMax = 16;                       // non-portable cluster size (sm_90+)
static constexpr int kClusterVertices = AVM_CLUSTER_VERTICES;

// Largest cooperative grid of the persistent kernel on the current device, capped by the work (0 = unavailable).
int persistent_grid(int V, bool per_cell) {
  int dev = 0, sms = 0, coop = 0, per_sm = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return 0;
  cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (!coop || sms <= 0) return 0;
  if (per_cell) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, persistent_steps_kernel<true, false>, kClusterBlock, 0);
  else cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, persistent_steps_kernel<false, false>, kClusterBlock, 0);
  if (per_sm < 1) return 0;
  const int want = V <= 512 ? 1 : cdiv(V, kClusterBlock), cap = sms * per_sm;     // tiny systems: one CTA, barriers are __syncthreads
  // up to kClusterVertices vertices the grid is one cluster of at most 16 CTAs (hardware barrier instead of an
  // arrival counter in L2); every thread then takes several vertices
  if (V > 512 && V <= kClusterVertices) { const int wc = cdiv(V, kClusterBlock); return wc < kClusterMax ? wc : kClusterMax; }
  return want < cap ? want : cap;
}

// n_steps timesteps in one cooperative launch; returns the number of launches (1), or -1 if the launch was refused.
int launch_persistent_steps(const Dev& d, const Consts& k, unsigned long long step0, int n_steps, int grid, cudaStream_t s) {
  Dev dd = d;
  Consts kk = k;
  kk.flag_dirty = 0; kk.clear_dirty = 0;
  int ns = n_steps;
  int one_cluster = 0;
  void* args[] = {(void*)&dd, (void*)&kk, (void*)&step0, (void*)&ns, (void*)&one_cluster};
  const void* fn = grid == 1 ? (k.per_cell ? (const void*)persistent_steps_kernel<true, true> : (const void*)persistent_steps_kernel<false, true>)
                             : (k.per_cell ? (const void*)persistent_steps_kernel<true, false> : (const void*)persistent_steps_kernel<false, false>);
  if (grid > 1 && grid <= kClusterMax && k.V <= kClusterVertices) {
    // the grid as one thread-block cluster: co-scheduled by construction, barriers in hardware
    one_cluster = 1;
    cudaFuncSetAttribute(fn, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3(kClusterBlock); cfg.dynamicSmemBytes = 0; cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)grid; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    if (cudaLaunchKernelExC(&cfg, fn, args) == cudaSuccess) return 1;
    cudaGetLastError();
    one_cluster = 0;                       // refused (cluster size not schedulable): the cooperative grid below
  }
  cudaMemsetAsync(&d.ctr->bar, 0, sizeof(unsigned int), s);
  if (cudaLaunchCooperativeKernel(fn, dim3((unsigned)grid), dim3(kClusterBlock), args, 0, s) != cudaSuccess) {
    cudaGetLastError();
    return -1;
  }
  return 1;
}

int launch_refresh_cells(const Dev& d, const Consts& k, cudaStream_t s) {
  if (k.per_cell) cell_update_kernel<false, true><<<cdiv(k.N, kCellBlock), kCellBlock, 0, s>>>(d, k, 0ull, 0u);
  else cell_update_kernel<false, false><<<cdiv(k.N, kCellBlock), kCellBlock, 0, s>>>(d, k, 0ull, 0u);
  return 1;
}

// leaves minkey all-idle and both candidate lists empty
int launch_t1_reset(const Dev& d, const Consts& k, cudaStream_t s) {
  t1_reset_kernel<<<kT1Grid, kT1Block, 0, s>>>(d, (unsigned)k.cap_a);
  zero_counts_kernel<<<1, 1, 0, s>>>(d);
  cudaMemsetAsync(d.dirty, 0, sizeof(unsigned int) * 2 * (size_t)k.nw, s);
  return 2;
}

int launch_t1_pass_only(const Dev& d, const Consts& k, cudaStream_t s) {
  int n = launch_t1_reset(d, k, s);
  detect_mark_kernel<<<cdiv(k.V, 256), 256, 0, s>>>(d, k, 0u, true);
  t1_flip_kernel<<<kT1Grid, kT1Block, 0, s>>>(d, k, 0u, true);
  n += 2;
  return n + launch_t1_reset(d, k, s);
}

int launch_t1_release(const Dev& d, const Consts& k, unsigned list, cudaStream_t s) {
  launch_chained(t1_release_kernel, kT1Grid, kT1Block, s, AVM_PDL != 0, d, k, list, (int)list);
  return 1;
}

int launch_t1_extra_pass(const Dev& d, const Consts& k, unsigned list_prev, unsigned list_new, unsigned stamp, cudaStream_t s) {
  const bool pdl = AVM_PDL != 0;     // part of the step's chain of dependent launches
  launch_chained(t1_release_kernel, kT1Grid, kT1Block, s, pdl, d, k, list_prev, (int)list_new);
  launch_chained(t1_local_detect_kernel, kT1Grid, kT1Block, s, pdl, d, k, list_prev, list_new, stamp);
  launch_chained(t1_flip_kernel, kT1Grid, kT1Block, s, pdl, d, k, list_new, true);
  return 3;
}

int launch_t1_debug(const Dev& d, const Consts& k, int* cand_pairs, int* win_pairs, long long capacity, cudaStream_t s) {
  int n = launch_t1_reset(d, k, s);
  detect_mark_kernel<<<cdiv(k.V, 256), 256, 0, s>>>(d, k, 0u, false);
  t1_debug_kernel<<<kT1Grid, kT1Block, 0, s>>>(d, cand_pairs, win_pairs, capacity);
  return n + 2;   // the caller reads the counters, then calls launch_t1_reset
}

int launch_compute_forces(const Dev& d, const Consts& k, double2* ap_scratch, double* force_user, double* ap_user, cudaStream_t s) {
  int n = 1;
  geometry_kernel<<<cdiv(k.N, 128), 128, 0, s>>>(d, k, ap_scratch, ap_user);
  if (force_user) { forces_kernel<<<cdiv(k.V, 256), 256, 0, s>>>(d, k, ap_scratch, force_user); ++n; }
  return n;
}

int launch_energy(const Dev& d, const Consts& k, double* partial, cudaStream_t s) {
  const int nb = 148 * 2;      // partial holds kObs * nb doubles
  observables_partial_kernel<<<nb, 256, 0, s>>>(d, k, partial);
  observables_final_kernel<<<1, 256, 0, s>>>(d, partial, nb, 1.0);
  return 2;
}

int launch_philox_words(unsigned long long seed, unsigned long long step, unsigned long long cell0, long long n,
                        uint32_t* out, cudaStream_t s) {
  if (n <= 0) return 0;
  philox_words_kernel<<<cdiv(n, 256), 256, 0, s>>>(seed, step, cell0, n, reinterpret_cast<uint4*>(out));
  return 1;
}

}  // namespace avm
