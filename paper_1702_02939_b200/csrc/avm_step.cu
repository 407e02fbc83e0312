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
//   T1 flips     (warp/candidate) rows a6+a7 (t1_try_flip): a candidate whose key is the minimum on
//                                  all four of its cells flips; the warp rewrites the four lists
//                                  cooperatively and refreshes the four cells' cached geometry.
//                                  Two-launch schedule (large systems): run by a few "flipper"
//                                  warps inside the NEXT step's force_move launch while the other
//                                  warps sweep.  Three-launch schedule: t1_flip_kernel.
//   repeated T1 passes (NEXT-1)    t1_release / t1_local_detect / t1_flip per extra pass.
// Geometry is thus evaluated once per step on the positions the forces of the following step
// act on; after a flip the records of its four cells are refreshed in place, so every force is
// computed from the geometry of the current topology exactly as in the paper's cycle.
#include <cstdio>
#include <cstdlib>
#include "avm_internal.cuh"

namespace avm {

static constexpr int kVertexBlock = 256;
static constexpr int kCellBlock = 128;
static constexpr int kT1Block = 128;
static constexpr int kT1Grid = 148 * 2;
static constexpr unsigned kFull = 0xffffffffu;

// tuning knobs (compile-time; the defaults are the measured best, profiles/)
#ifndef AVM_FM_PF
#define AVM_FM_PF 1        // force_move: L2 prefetch distance in grid sweeps (0 = off)
#endif
#ifndef AVM_PDL
#define AVM_PDL 1          // chain the step's kernels with programmatic dependent launch
#endif
#ifndef AVM_CU_MINB
#define AVM_CU_MINB 8      // cell pass: resident CTAs per SM asked of the compiler (64 registers; measured best of 7..11)
#endif
#ifndef AVM_FM_COOP
#define AVM_FM_COOP 0       // launch the fused force_move as a cooperative grid (not needed: work is claimed, see flipper_work)
#endif
#ifndef AVM_FM_MINB
#define AVM_FM_MINB 3      // force_move: minimum resident CTAs per SM asked of the compiler
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
// one 32-byte record with a single 256-bit load (LDG.E.256, sm_100)
__device__ __forceinline__ CellRec ld_rec(const CellRec* p) {
  CellRec r;
  asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(r.a), "=d"(r.p), "=d"(r.nx), "=d"(r.ny) : "l"(p));
  return r;
}
__device__ __forceinline__ void st_rec(CellRec* p, const CellRec& r) {
  asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(r.a), "d"(r.p), "d"(r.nx), "d"(r.ny) : "memory");
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

struct VertexIn { double2 h; int n0, n1, n2, c0, c1, c2; };
__device__ __forceinline__ VertexIn load_vertex(const Dev& d, const Consts& k, int v) {
  VertexIn in;
  in.h = __ldg(d.pos + v);
  in.n0 = ld_stream(d.vn + v); in.n1 = ld_stream(d.vn + k.Vs + v); in.n2 = ld_stream(d.vn + 2 * k.Vs + v);
  in.c0 = ld_stream(d.vc + v); in.c1 = ld_stream(d.vc + k.Vs + v); in.c2 = ld_stream(d.vc + 2 * k.Vs + v);
  return in;
}

// Eq. 4: dh/dt = mu F + (v0/3) sum of the three unit directors (R5), directors of the start of
// the step (R7); explicit Euler; wrap into the box (R13).
__device__ __forceinline__ void move_vertex(const Dev& d, const Consts& k, int v, const double2 h, const double2 q0,
                                            const double2 q1, const double2 q2, const CellRec& c0, const CellRec& c1,
                                            const CellRec& c2) {
  const double2 f = vertex_force(h, q0, q1, q2, c0, c1, c2, k);
  const double vx = __fma_rn(k.mu, f.x, __dmul_rn(k.v0_3, __dadd_rn(__dadd_rn(c0.nx, c1.nx), c2.nx)));
  const double vy = __fma_rn(k.mu, f.y, __dmul_rn(k.v0_3, __dadd_rn(__dadd_rn(c0.ny, c1.ny), c2.ny)));
  double x = __fma_rn(k.dt, vx, h.x), y = __fma_rn(k.dt, vy, h.y);
  // negative, >= L (conservatively) and non-finite values all have a large unsigned high word
  if ((hi_word(x) >= hi_word(k.Lx)) | (hi_word(y) >= hi_word(k.Ly))) {
    x = wrap_box(x, k.Lx); y = wrap_box(y, k.Ly);
    if (!(isfinite(x) && isfinite(y))) atomicOr((unsigned long long*)&d.ctr->error, 1ull);
  }
  d.pos_next[v] = make_double2(x, y);
}

// the same vertex update with every input read from L2 (after another warp of this launch
// rewrote the neighbourhood: L1 may hold stale lines)
__device__ __noinline__ void move_vertex_coherent(const Dev& d, const Consts& k, int v) {
  const double2 h = __ldcg(d.pos + v);
  double2 q[3];
  CellRec c[3];
#pragma unroll
  for (int s = 0; s < 3; ++s) {
    q[s] = __ldcg(d.pos + __ldcg(d.vn + s * k.Vs + v));
    const double2* r = reinterpret_cast<const double2*>(d.rec + __ldcg(d.vc + s * k.Vs + v));
    const double2 ap = __ldcg(r), nn = __ldcg(r + 1);
    c[s].a = ap.x; c[s].p = ap.y; c[s].nx = nn.x; c[s].ny = nn.y;
  }
  move_vertex(d, k, v, h, q[0], q[1], q[2], c[0], c[1], c[2]);
}

__device__ __forceinline__ unsigned int ld_volatile(const unsigned int* p) {
  unsigned int x;
  asm volatile("ld.volatile.global.u32 %0, [%1];" : "=r"(x) : "l"(p) : "memory");
  return x;
}

__device__ __noinline__ bool t1_try_flip(const Dev& d, const Consts& k, const Cand& c, const int lane);

// The sweep of one thread over vertices first, first + step_v, ...  kSkipDirty: vertices
// flagged in d.dirty are left to the flippers.
template <bool kSkipDirty>
__device__ __forceinline__ void sweep(const Dev& d, const Consts& k, const int first, const int step_v, const int lane) {
  if (first >= k.V) return;
  int v = first;
  VertexIn in = load_vertex(d, k, v);
  unsigned dw = kSkipDirty ? __ldg(d.dirty + (v >> 5)) : 0u;
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
      const double2 q0 = __ldg(d.pos + in.n0), q1 = __ldg(d.pos + in.n1), q2 = __ldg(d.pos + in.n2);
      const CellRec c0 = ld_rec(d.rec + in.c0), c1 = ld_rec(d.rec + in.c1), c2 = ld_rec(d.rec + in.c2);
      const double2 h = in.h;
      if (AVM_FM_REGPF && vnext < k.V) { in = load_vertex(d, k, vnext); if (kSkipDirty) dw = __ldg(d.dirty + (vnext >> 5)); }
      move_vertex(d, k, v, h, q0, q1, q2, c0, c1, c2);
    } else if (AVM_FM_REGPF && vnext < k.V) {
      in = load_vertex(d, k, vnext);
      dw = __ldg(d.dirty + (vnext >> 5));
    }
    if (vnext >= k.V) break;
    v = vnext;
    if (!AVM_FM_REGPF) { in = load_vertex(d, k, v); if (kSkipDirty) dw = __ldg(d.dirty + (v >> 5)); }
  }
}

// Rows a6 + a7 of the previous step inside the fused force_move launch, run by the "flipper"
// warps (the first F warps of the grid, which take no share of the sweep).  Work is CLAIMED with
// atomic counters, so a candidate always belongs to a warp that is running: the wait below can
// never depend on a CTA that has not been scheduled yet (no co-residency assumption).
//   1. claim candidates one by one; decide and flip each (t1_try_flip);
//   2. wait until every candidate has been decided (flip_done == prev);
//   3. claim candidates again: move the flagged vertices of the candidate's four cells with
//      loads that bypass L1 (whoever clears a vertex's bit moves it) and release the cells'
//      minimum keys (row a6).
__device__ __noinline__ void flipper_flips(const Dev& d, const Consts& k, const unsigned prev, const int lane) {
  unsigned mine = 0, flips = 0;
  for (;;) {
    unsigned i = 0;
    if (lane == 0) i = atomicAdd(&d.ctr->next_cand, 1u);
    i = __shfl_sync(kFull, i, 0);
    if (i >= prev) break;
    const Cand c = d.cand[i];
    if (t1_try_flip(d, k, c, lane)) ++flips;
    ++mine;
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

__device__ __noinline__ void flipper_moves(const Dev& d, const Consts& k, const unsigned prev, const int lane) {
  while (ld_volatile(&d.ctr->flip_done) < prev) __nanosleep(64);
  __threadfence();
  // rows of up to 16 entries: two rows per pass (half a warp each), else one row per pass
  const bool two = k.S <= 16;
  const int half = two ? lane >> 4 : 0, j = two ? lane & 15 : lane;
  for (;;) {
    unsigned i = 0;
    if (lane == 0) i = atomicAdd(&d.ctr->next_quad, 1u);
    i = __shfl_sync(kFull, i, 0);
    if (i >= prev) break;
    const Cand c = d.cand[i];
    const int quad[4] = {c.cL, c.cR, c.cE1, c.cE2};
#pragma unroll 1
    for (int t0 = 0; t0 < 4; t0 += (two ? 2 : 1)) {
      const int cell = quad[t0 + half];
      // the entry is loaded whatever the row length is (padding repeats entry 0): no dependent load
      const int n = __ldcg(d.cvn + cell);
      const int u = __ldcg(reinterpret_cast<const int*>(d.cv + (size_t)(j >> 2) * k.N + cell) + (j & 3));
      if (j < n) {
        const unsigned bit = 1u << (u & 31);
        if (atomicAnd(&d.dirty[u >> 5], ~bit) & bit) move_vertex_coherent(d, k, u);
      }
    }
    if (lane < 4) d.minkey[quad[lane & 3]] = ~0ull;
  }
}

// Persistent grid-stride kernel: each thread keeps the streaming loads of its NEXT vertex in
// flight while it gathers and computes the current one.
//
// kFused also carries rows a6 + a7 of the PREVIOUS step (flipper_flips / flipper_moves above):
// a few warps decide and flip that step's candidates while all other warps already move
// vertices.  A vertex whose inputs a flip may rewrite has its bit set in d.dirty (the marking
// thread flagged every vertex of the candidate's four cells); the sweep skips it and a flipper
// moves it once every candidate has been decided.  The latency-bound flips thus overlap the
// gather-bound sweep and the step needs no third launch.
template <bool kFused>
__global__ void __launch_bounds__(kVertexBlock, AVM_FM_MINB)
force_move_kernel(const __grid_constant__ Dev d, const __grid_constant__ Consts k, const unsigned parity) {
  pdl_launch_dependents();
  pdl_wait();
  const int tid = blockIdx.x * kVertexBlock + threadIdx.x;
  const int stride = gridDim.x * kVertexBlock;
  const int lane = threadIdx.x & 31;
  const unsigned prev = min(d.ctr->n_cand[parity ^ 1u], (unsigned)k.cap_a);
  const unsigned gwarp = (unsigned)tid >> 5, nwarps = (unsigned)stride >> 5;
  if (tid == 0) d.ctr->n_cand[parity] = 0;
  if (kFused) {
    if (tid == 0 && prev) atomicAdd((unsigned long long*)&d.ctr->t1_candidates, (unsigned long long)prev);
    if (2u * prev <= nwarps) {
      // few candidates: the first `prev` warps only flip (they would start the sweep late and
      // finish it last), all others only sweep
      if (gwarp < prev) {
        flipper_flips(d, k, prev, lane);
        flipper_moves(d, k, prev, lane);
      } else {
        const int first = (int)(gwarp - prev) * 32 + lane, step_v = (int)(nwarps - prev) * 32;
        if (prev) sweep<true>(d, k, first, step_v, lane);
        else sweep<false>(d, k, first, step_v, lane);
      }
    } else {
      // many candidates (the burst after a random start, T1-heavy regimes): every warp flips,
      // then sweeps its share, then moves flagged vertices
      flipper_flips(d, k, prev, lane);
      sweep<true>(d, k, tid, stride, lane);
      flipper_moves(d, k, prev, lane);
    }
  } else {
    // the previous step's T1 candidates are done: clear their cells' minimum keys (row a6)
    for (unsigned i = tid; i < prev; i += stride) {
      const Cand c = d.cand[i];
      d.minkey[c.cL] = ~0ull; d.minkey[c.cR] = ~0ull; d.minkey[c.cE1] = ~0ull; d.minkey[c.cE2] = ~0ull;
    }
    sweep<false>(d, k, tid, stride, lane);
  }
}

// ---------------------------------------------------------------------------------------------
// rows a5 (eligibility, R10) + a6 (marking half of the conflict rule, R11) for ONE short edge,
// run by the thread that found it.  (va, vb) are current vertex indices.  Cold path.
// ---------------------------------------------------------------------------------------------
__device__ __noinline__ void t1_mark_edge(const Dev& d, const Consts& k, int va, int vb, unsigned parity, bool count_stats) {
  // The marking thread delays the end of the cell pass when it sits in the last wave, so its
  // loads are issued in two batches of independent loads instead of a chain of five.
  // ---- batch 1: everything known from (va, vb) ----
  const double2 ha = d.pos[va], hb = d.pos[vb];
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
#pragma unroll
  for (int t = 0; t < 4; ++t) { nq[t] = d.cvn[quad[t]]; q[t][0] = d.cv[quad[t]]; q[t][1] = d.cv[(size_t)k.N + quad[t]]; }
  const int x1s1 = d.vn[k.Vs + x1], x1s2 = d.vn[2 * k.Vs + x1], x2s1 = d.vn[k.Vs + x2], x2s2 = d.vn[2 * k.Vs + x2];
  if (!(nq[0] > 3 && nq[1] > 3)) return;                       // no 2-gons (T2 absent)
  if (!(nq[2] < k.S && nq[3] < k.S)) {                         // row would exceed the stride
    if (count_stats) {
      atomicAdd((unsigned long long*)&d.ctr->overflow_rejects, 1ull);
      atomicOr((unsigned long long*)&d.ctr->error, 2ull);
    }
    return;
  }
  Cand cd;
  cd.v1 = v1; cd.v2 = v2; cd.k1 = k1; cd.k2 = k2;
  cd.cL = cL; cd.cR = cR; cd.cE1 = cE1; cd.cE2 = cE2;
  cd.key = ((unsigned long long)t1 << 32) | t2;
  cd.x1 = x1; cd.y1 = y1; cd.x2 = x2; cd.y2 = y2;
  cd.sx1 = x1s1 == v1 ? 1 : x1s2 == v1 ? 2 : 0;
  cd.sx2 = x2s1 == v2 ? 1 : x2s2 == v2 ? 2 : 0;
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
  if (count_stats && k.flag_dirty) {
#pragma unroll
    for (int t = 0; t < 4; ++t) {
      const int e[8] = {q[t][0].x, q[t][0].y, q[t][0].z, q[t][0].w, q[t][1].x, q[t][1].y, q[t][1].z, q[t][1].w};
#pragma unroll
      for (int j = 0; j < 8; ++j) atomicOr(&d.dirty[e[j] >> 5], 1u << (e[j] & 31));   // padding repeats entry 0
      for (int j = 8; j < nq[t]; ++j) {
        const int u = row_entry(d.cv, k.N, quad[t], j);
        atomicOr(&d.dirty[u >> 5], 1u << (u & 31));
      }
    }
  }
}

// The geometry pass flagged edges of cell c (bit j-1 = the edge ending at row entry j, j = n
// being the closing edge) as possibly short.  Each edge is seen by its two cells in opposite
// directions: it is reported from the cell that traverses it from the smaller to the larger
// (current) vertex index.
__device__ __noinline__ void t1_report_cell(const Dev& d, const Consts& k, int c, int n, unsigned smask, unsigned parity) {
  while (smask) {
    const int j = __ffs(smask);     // edge (j-1) -> (j mod n)
    smask &= smask - 1u;
    const int va = row_entry(d.cv, k.N, c, j - 1), vb = row_entry(d.cv, k.N, c, j == n ? 0 : j);
    if (va < vb) t1_mark_edge(d, k, va, vb, parity, true);
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
template <bool kStep, bool kPerCell>
__global__ void __launch_bounds__(kCellBlock, AVM_CU_MINB)
cell_update_kernel(const __grid_constant__ Dev d, const __grid_constant__ Consts k, const unsigned long long step,
                   const unsigned parity) {
  pdl_launch_dependents();
  pdl_wait();
  const int gid = blockIdx.x * kCellBlock + threadIdx.x;
  if (kStep && gid == 0) { d.ctr->flip_done = 0; d.ctr->next_cand = 0; d.ctr->next_quad = 0; }   // the previous list is long done
  const bool valid = gid < k.N;
  const int c = valid ? k.N - 1 - gid : 0;
  const double2* __restrict__ pos = d.pos;
  const int n = valid ? ld_stream(d.cvn + c) : 0;
  const int4 qa = ld_stream(d.cv + c), qb = ld_stream(d.cv + k.N + c);
  const int e[8] = {qa.x, qa.y, qa.z, qa.w, qb.x, qb.y, qb.z, qb.w};
  double th = ld_stream(d.theta + c);
  const unsigned int tag = (unsigned int)ld_stream(d.ctag + c);
  double2 h[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) h[j] = __ldg(pos + e[j]);   // padding entries repeat entry 0: r = 0, no predicate
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
      const int4 qq = d.cv[(size_t)q * k.N + c];
      const int ee[4] = {qq.x, qq.y, qq.z, qq.w};
      double2 hh[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        hh[i] = h[0];
        if (j0 + i < n) hh[i] = __ldg(pos + ee[i]);
      }
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        if (j0 + i < n) {
          const double x = min_image(__dsub_rn(hh[i].x, h[0].x), k.Lx, k.hLx);
          const double y = min_image(__dsub_rn(hh[i].y, h[0].y), k.Ly, k.hLy);
          const double l2 = geom_edge(rxp, ryp, x, y, acc, per);
          if (kStep && hi_word(l2) <= hlc) smask |= 1u << (j0 + i - 1);
          rxp = x; ryp = y;
        }
      }
    }
  }
  {  // closing edge of an n >= 8 cell (an exact no-op for smaller ones, which closed above)
    const double l2 = geom_edge(rxp, ryp, 0.0, 0.0, acc, per);
    if (kStep && hi_word(l2) <= hlc) smask |= 1u << ((n > 8 ? n : 8) - 1);
  }
  if (!valid) return;
  CellRec r;
  const double2 tg = kPerCell ? d.tgt[c] : make_double2(k.A0, k.P0);   // Eq. 1 per cell (NEXT-4) / Eq. A1
  r.a = k.KA2 * (__dmul_rn(0.5, acc) - tg.x);
  r.p = k.KP2 * (per - tg.y);
  r.nx = cs; r.ny = sn;
  st_rec(d.rec + c, r);
  smask &= n >= 32 ? ~0u : (1u << n) - 1u;     // edges beyond the closing one are padding
  if (kStep && smask) t1_report_cell(d, k, c, n, smask, parity);
}

// Detection alone (test hooks avm_t1_pass / avm_debug_t1): thread per vertex, edge owned by the
// smaller current index.
__global__ void detect_mark_kernel(const __grid_constant__ Dev d, const __grid_constant__ Consts k, const unsigned parity,
                                   const bool count_stats) {
  const int v = blockIdx.x * blockDim.x + threadIdx.x;
  if (v >= k.V) return;
  const double2 h = d.pos[v];
  for (int s = 0; s < 3; ++s) {
    const int w = d.vn[s * k.Vs + v];
    if (v < w) {
      // cheap pre-test; t1_mark_edge repeats the canonical one
      const double2 q = d.pos[w];
      const double dx = min_image(q.x - h.x, k.Lx, k.hLx), dy = min_image(q.y - h.y, k.Ly, k.hLy);
      if (dx * dx + dy * dy < k.lc2) t1_mark_edge(d, k, v, w, parity, count_stats);
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
      const double2 hu = d.pos[u];
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
        const double2 hw = d.pos[wv];
        const double dx = min_image(hw.x - hu.x, k.Lx, k.hLx), dy = min_image(hw.y - hu.y, k.Ly, k.hLy);
        if (dx * dx + dy * dy < k.lc2) t1_mark_edge(d, k, owner, other, list_new, false);
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// rows a6 (deciding half) + a7: flip + rewrite (R9 geometry, R12 lists), one WARP per candidate.
// A candidate flips iff its key is the minimum recorded on all four of its cells (R11); winners
// therefore own disjoint cell quadruples and every word written below belongs to a vertex or row
// inside the winner's own quadruple.  minkey is only read here (cleared by the next force_move).
// ---------------------------------------------------------------------------------------------
// One candidate, one warp: decide (R11) and, if it wins, flip and rewrite (R9, R12).  Returns
// whether the edge flipped.  Used by the stand-alone T1 kernel and by force_move's fused prologue.
__device__ __noinline__ bool t1_try_flip(const Dev& d, const Consts& k, const Cand& c, const int lane) {
  const int cells[4] = {c.cL, c.cR, c.cE1, c.cE2};
  const int l4 = lane & 3;
  // ---- everything is read before anything is written; the loads below are independent of
  // one another (the marking thread decoded the neighbourhood), so the minimum-key test
  // costs no extra round trip ----
  const unsigned long long mk = d.minkey[l4 == 0 ? c.cL : l4 == 1 ? c.cR : l4 == 2 ? c.cE1 : c.cE2];
  const int v1 = c.v1, v2 = c.v2, k1 = c.k1, k2 = c.k2;
  const int a1 = (k1 + 1) % 3, b1 = (k1 + 2) % 3, a2 = (k2 + 1) % 3, b2 = (k2 + 2) % 3;
  const double2 h1 = d.pos[v1], h2 = d.pos[v2];
  const int x1 = c.x1, y1 = c.y1, x2 = c.x2, y2 = c.y2;
  int row[4], nrow[4];
#pragma unroll
  for (int t = 0; t < 4; ++t) {
    nrow[t] = d.cvn[cells[t]];
    row[t] = row_entry(d.cv, k.N, cells[t], lane < k.S ? lane : 0);
  }
  if (!__all_sync(kFull, mk == c.key)) return false;
  // ---- geometry: rigid counter-clockwise quarter turn about the midpoint, new length 1.5 l_c (R9)
  const double dx = min_image(h2.x - h1.x, k.Lx, k.hLx), dy = min_image(h2.y - h1.y, k.Ly, k.hLy);
  const double l = sqrt(dx * dx + dy * dy);
  const double mx = h1.x + 0.5 * dx, my = h1.y + 0.5 * dy;
  double px = 0.0, py = 1.0;
  if (l > 0.0) { px = -dy / l; py = dx / l; }
  const double half = 0.75 * k.lc;
  const double2 n2 = make_double2(wrap_box(mx + half * px, k.Lx), wrap_box(my + half * py, k.Ly));
  const double2 n1 = make_double2(wrap_box(mx - half * px, k.Lx), wrap_box(my - half * py, k.Ly));
  if (lane == 0) {
    d.pos[v2] = n2;
    d.pos[v1] = n1;
    // lists: u = ([w, x, y]; [C0, C1, C2]) cyclic from the partner slot
    //     -> ([w, y, z]; [C1, C2, C']), z = partner's old x, C' = partner's old C1 (R12)
    d.vn[a1 * k.Vs + v1] = y1; d.vn[b1 * k.Vs + v1] = x2;
    d.vc[k1 * k.Vs + v1] = c.cE1; d.vc[a1 * k.Vs + v1] = c.cR; d.vc[b1 * k.Vs + v1] = c.cE2;
    d.vn[a2 * k.Vs + v2] = y2; d.vn[b2 * k.Vs + v2] = x1;
    d.vc[k2 * k.Vs + v2] = c.cE2; d.vc[a2 * k.Vs + v2] = c.cL; d.vc[b2 * k.Vs + v2] = c.cE1;
  }
  // outer vertices: x1 was joined to v1 and is now joined to v2 (same slot); x2 likewise
  if (lane == 1) d.vn[c.sx1 * k.Vs + x1] = v2;
  if (lane == 2) d.vn[c.sx2 * k.Vs + x2] = v1;
  // rows (lane = row entry): L deletes v1, R deletes v2 (later entries shift down); E1 inserts
  // v2 immediately after v1, E2 inserts v1 immediately after v2 (later entries shift up).
  // The new rows are formed in registers, written back, and reused by the refresh below.
  int nnew[4];
#pragma unroll
  for (int t = 0; t < 4; ++t) {
    int r = row[t];
    if (t < 2) {
      const int victim = t == 0 ? v1 : v2;
      const int p = __ffs(__ballot_sync(kFull, lane < nrow[t] && r == victim)) - 1;
      const int nxt = __shfl_down_sync(kFull, r, 1);
      nnew[t] = nrow[t] - 1;
      if (lane >= p) r = nxt;
    } else {
      const int after = t == 2 ? v1 : v2, ins = t == 2 ? v2 : v1;
      const int p = __ffs(__ballot_sync(kFull, lane < nrow[t] && r == after)) - 1;
      const int prv = __shfl_up_sync(kFull, r, 1);
      nnew[t] = nrow[t] + 1;
      if (lane > p) r = lane == p + 1 ? ins : prv;
    }
    const int r0 = __shfl_sync(kFull, r, 0);
    if (lane >= nnew[t]) r = r0;                         // padding repeats entry 0
    if (lane < k.S && r != row[t]) row_entry(d.cv, k.N, cells[t], lane) = r;
    if (lane == 0) d.cvn[cells[t]] = nnew[t];
    row[t] = r;
  }
  // refresh the cached geometry of the four cells (directors unchanged): every lane fetches
  // the position of "its" entry of each row (v1 and v2 take their new positions from
  // registers), then the warp runs the same serial sum as the per-step pass, so that a resumed
  // run reproduces these records bit for bit.  Lane t keeps cell t's result.
  double2 hr[4];
#pragma unroll
  for (int t = 0; t < 4; ++t) {
    hr[t] = make_double2(0.0, 0.0);
    const int v = row[t];
    if (lane < nnew[t]) hr[t] = v == v1 ? n1 : v == v2 ? n2 : d.pos[v];
  }
  // lane j holds entry j of each row: unwrapped position (ux, uy) and the length of the edge
  // that ENDS at entry j (lane 0: the closing edge), computed in parallel with geom_edge's
  // arithmetic; the order-dependent sums then run as four interleaved serial chains.
  double ux[4], uy[4], sl[4];
  int nmax = 0;
#pragma unroll
  for (int t = 0; t < 4; ++t) {
    const double h0x = __shfl_sync(kFull, hr[t].x, 0), h0y = __shfl_sync(kFull, hr[t].y, 0);
    ux[t] = min_image(__dsub_rn(hr[t].x, h0x), k.Lx, k.hLx);
    uy[t] = min_image(__dsub_rn(hr[t].y, h0y), k.Ly, k.hLy);
    const int prev = lane == 0 ? nnew[t] - 1 : lane - 1;
    const double pxv = __shfl_sync(kFull, ux[t], prev), pyv = __shfl_sync(kFull, uy[t], prev);
    const double dx = __dsub_rn(ux[t], pxv), dy = __dsub_rn(uy[t], pyv);
    sl[t] = sqrt_pos(__fma_rn(dx, dx, __fma_rn(dy, dy, kTiny)));
    nmax = max(nmax, nnew[t]);
  }
  double rxp[4] = {0.0, 0.0, 0.0, 0.0}, ryp[4] = {0.0, 0.0, 0.0, 0.0}, acc[4] = {0.0, 0.0, 0.0, 0.0},
         per[4] = {0.0, 0.0, 0.0, 0.0};
  for (int j = 1; j <= nmax; ++j) {
#pragma unroll
    for (int t = 0; t < 4; ++t) {
      if (j <= nnew[t]) {                          // warp-uniform
        const int src = j < nnew[t] ? j : 0;       // j == n: the closing edge back to entry 0 (r = 0)
        const double x = __shfl_sync(kFull, ux[t], src), y = __shfl_sync(kFull, uy[t], src);
        const double l = __shfl_sync(kFull, sl[t], src);
        acc[t] = __fma_rn(rxp[t], y, acc[t]);
        acc[t] = __fma_rn(-ryp[t], x, acc[t]);
        per[t] = __dadd_rn(per[t], l);
        rxp[t] = x; ryp[t] = y;
      }
    }
  }
  double myA = 0.0, myP = 0.0;
#pragma unroll
  for (int t = 0; t < 4; ++t)
    if (lane == t) { myA = __dmul_rn(0.5, acc[t]); myP = per[t]; }
  if (lane < 4) {
    const int cc = cells[lane == 0 ? 0 : lane == 1 ? 1 : lane == 2 ? 2 : 3];
    const double2 tg = cell_targets(d, k, cc);
    d.rec[cc].a = k.KA2 * (myA - tg.x);
    d.rec[cc].p = k.KP2 * (myP - tg.y);
  }
  __syncwarp();
  return true;
}

__global__ void __launch_bounds__(kT1Block)
t1_flip_kernel(const __grid_constant__ Dev d, const __grid_constant__ Consts k, const unsigned parity, const bool count_stats) {
  pdl_launch_dependents();
  pdl_wait();
  const unsigned int n_cand = min(d.ctr->n_cand[parity], list_cap(k, parity));
  const Cand* __restrict__ list = list_base(d, k, parity);
  const int lane = threadIdx.x & 31;
  const unsigned gwarp = (blockIdx.x * kT1Block + threadIdx.x) >> 5, nwarps = (gridDim.x * kT1Block) >> 5;
  if (count_stats && gwarp == 0 && lane == 0 && n_cand) atomicAdd((unsigned long long*)&d.ctr->t1_candidates, (unsigned long long)n_cand);
  unsigned int flips = 0, blocked = 0;
  for (unsigned int i = gwarp; i < n_cand; i += nwarps) {
    const Cand c = list[i];
    if (t1_try_flip(d, k, c, lane)) ++flips; else ++blocked;
  }
  if (count_stats && lane == 0) {
    if (flips) atomicAdd((unsigned long long*)&d.ctr->t1_flips, (unsigned long long)flips);
    if (blocked) atomicAdd((unsigned long long*)&d.ctr->t1_blocked, (unsigned long long)blocked);
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
__global__ void zero_counts_kernel(const Dev d) { d.ctr->n_cand[0] = 0; d.ctr->n_cand[1] = 0; d.ctr->n_cand[2] = 0; d.ctr->n_cand[3] = 0; d.ctr->n_win = 0; d.ctr->flip_done = 0; d.ctr->next_cand = 0; d.ctr->next_quad = 0; }

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
  const double2 h = d.pos[v];
  CellRec c[3];
  double2 q[3];
#pragma unroll
  for (int s = 0; s < 3; ++s) {
    q[s] = d.pos[d.vn[s * k.Vs + v]];
    const int cell = d.vc[s * k.Vs + v];
    const double2 a = ap[cell], tg = cell_targets(d, k, cell);
    c[s].a = k.KA2 * (a.x - tg.x); c[s].p = k.KP2 * (a.y - tg.y); c[s].nx = 0.0; c[s].ny = 0.0;
  }
  const double2 f = vertex_force(h, q[0], q[1], q[2], c[0], c[1], c[2], k);
  const int t = d.vtag[v];
  force_user[2 * t] = f.x; force_user[2 * t + 1] = f.y;
}

// Observables of the current state (NEXT-2): energy, Eq. 1 / A1, and the
// per-cell statistics a user of the model measures (shape index P / sqrt(A), area moments).
// Slots: 0 energy, 1 sum A, 2 sum P, 3 sum P/sqrt(A) over cells with A > 0, 4 number of cells with
// A <= 0, 5 sum A^2, 6 min A, 7 max A.  Block partials in a fixed order, finished by one block
// (deterministic, no floating-point atomics).
static constexpr int kObs = 8;
__device__ __forceinline__ double obs_combine(int slot, double a, double b) {
  return slot < 6 ? a + b : slot == 6 ? fmin(a, b) : fmax(a, b);
}
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
  double x[kObs] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 1.0e300, -1.0e300};
  for (int c = blockIdx.x * 256 + threadIdx.x; c < k.N; c += gridDim.x * 256) {
    double A, P;
    cell_area_perimeter(d.pos, d.cv, c, d.cvn[c], k, A, P);
    const double2 tg = cell_targets(d, k, c);
    x[0] += k.KA * (A - tg.x) * (A - tg.x) + k.KP * (P - tg.y) * (P - tg.y);
    x[1] += A; x[2] += P;
    if (A > 0.0) x[3] += P / sqrt(A); else x[4] += 1.0;
    x[5] += A * A;
    x[6] = fmin(x[6], A); x[7] = fmax(x[7], A);
  }
  obs_block_reduce(x, sm);
  if (threadIdx.x < kObs) partial[(size_t)threadIdx.x * gridDim.x + blockIdx.x] = sm[threadIdx.x][0];
}
__global__ void __launch_bounds__(256)
observables_final_kernel(const Dev d, const double* __restrict__ partial, int n) {
  __shared__ double sm[kObs][256];
  double x[kObs] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 1.0e300, -1.0e300};
  for (int i = threadIdx.x; i < n; i += 256)
#pragma unroll
    for (int q = 0; q < kObs; ++q) x[q] = obs_combine(q, x[q], partial[(size_t)q * n + i]);
  obs_block_reduce(x, sm);
  if (threadIdx.x < kObs) d.ctr->obs[threadIdx.x] = sm[threadIdx.x][0];
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

static int force_move_grid(const Consts& k) {
  // persistent: a whole number of CTAs per SM (148 SMs), never more CTAs than there is work
  static int per_sm = 0;
  if (!per_sm) {
    int a = 0, b = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&a, force_move_kernel<true>, kVertexBlock, 0);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, force_move_kernel<false>, kVertexBlock, 0);
    per_sm = a < b ? a : b;
    if (per_sm < 1) per_sm = 1;
  }
  const int want = cdiv(k.V, kVertexBlock);
  const int cap = 148 * per_sm;
  return want < cap ? want : cap;
}

// Launch with the programmatic-stream-serialization attribute (see pdl_wait above) and,
// optionally, as a cooperative grid (every CTA resident: force_move<true> spins on a counter
// that other CTAs advance).
template <typename... KArgs, typename... Args>
static cudaError_t launch_chained(void (*kernel)(KArgs...), int grid, int block, cudaStream_t s, bool pdl, bool coop,
                                  Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)block); cfg.dynamicSmemBytes = 0; cfg.stream = s;
  cudaLaunchAttribute attr[2];
  int na = 0;
  if (pdl) { attr[na].id = cudaLaunchAttributeProgrammaticStreamSerialization; attr[na].val.programmaticStreamSerializationAllowed = 1; ++na; }
  if (coop) { attr[na].id = cudaLaunchAttributeCooperative; attr[na].val.cooperative = 1; ++na; }
  cfg.attrs = attr; cfg.numAttrs = (unsigned)na;
  return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// One timestep.  d.pos = positions at the start of the step, d.pos_next = buffer for the moved
// positions (the caller swaps them afterwards).
//   fused = true : two launches; the T1 flips of the PREVIOUS step ride in force_move's
//                  prologue, those of this step stay pending (launch_t1_flush applies them).
//   fused = false: three launches, each step complete on return (also the per-kernel timing mode).
// ev (optional, AVM_K_COUNT+1 events): recorded before/after each kernel by avm_step_profile.
int launch_step(const Dev& d, const Consts& k, unsigned long long step, cudaStream_t s, cudaEvent_t* ev, bool fused) {
  const unsigned parity = (unsigned)(step & 1ull);
  if (ev) cudaEventRecord(ev[0], s);
  const bool pdl = AVM_PDL && ev == nullptr;   // events between the kernels would break the chain anyway
  static int coop_pdl_ok = 1;                  // cooperative + programmatic launch accepted by this driver?
  if (fused) {
    cudaError_t e = cudaErrorUnknown;
    if (pdl && coop_pdl_ok) {
      e = launch_chained(force_move_kernel<true>, force_move_grid(k), kVertexBlock, s, true, AVM_FM_COOP != 0, d, k, parity);
      if (e != cudaSuccess) { coop_pdl_ok = 0; cudaGetLastError(); if (getenv("AVM_B200_DEBUG")) fprintf(stderr, "avm: cooperative+programmatic launch rejected\n"); }
    }
    if (e != cudaSuccess) e = launch_chained(force_move_kernel<true>, force_move_grid(k), kVertexBlock, s, false, AVM_FM_COOP != 0, d, k, parity);
    if (e != cudaSuccess) return -1;           // the caller falls back to the unfused schedule
  } else {
    launch_chained(force_move_kernel<false>, force_move_grid(k), kVertexBlock, s, pdl, false, d, k, parity);
  }
  if (ev) cudaEventRecord(ev[1], s);
  Dev m = d;                      // from here on the moved positions are "the" positions
  m.pos = d.pos_next; m.pos_next = d.pos;
  if (k.per_cell) launch_chained(cell_update_kernel<true, true>, cdiv(k.N, kCellBlock), kCellBlock, s, pdl, false, m, k, step, parity);
  else launch_chained(cell_update_kernel<true, false>, cdiv(k.N, kCellBlock), kCellBlock, s, pdl, false, m, k, step, parity);
  if (ev) cudaEventRecord(ev[2], s);
  if (!fused) launch_chained(t1_flip_kernel, kT1Grid, kT1Block, s, pdl, false, m, k, parity, true);
  if (ev) cudaEventRecord(ev[3], s);
  return fused ? 2 : 3;
}

// Applies the flips a fused step left pending (d = the state after that step) and leaves the T1
// work lists idle, so that any other entry point sees a complete step.
int launch_t1_flush(const Dev& d, const Consts& k, unsigned long long last_step, cudaStream_t s) {
  t1_flip_kernel<<<kT1Grid, kT1Block, 0, s>>>(d, k, (unsigned)(last_step & 1ull), true);
  return 1 + launch_t1_reset(d, k, s);
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
  cudaMemsetAsync(d.dirty, 0, sizeof(unsigned int) * (size_t)((k.V + 31) / 32), s);
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
  launch_chained(t1_release_kernel, kT1Grid, kT1Block, s, AVM_PDL != 0, false, d, k, list, (int)list);
  return 1;
}

int launch_t1_extra_pass(const Dev& d, const Consts& k, unsigned list_prev, unsigned list_new, unsigned stamp, cudaStream_t s) {
  const bool pdl = AVM_PDL != 0;     // part of the step's chain of dependent launches
  launch_chained(t1_release_kernel, kT1Grid, kT1Block, s, pdl, false, d, k, list_prev, (int)list_new);
  launch_chained(t1_local_detect_kernel, kT1Grid, kT1Block, s, pdl, false, d, k, list_prev, list_new, stamp);
  launch_chained(t1_flip_kernel, kT1Grid, kT1Block, s, pdl, false, d, k, list_new, true);
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
  observables_final_kernel<<<1, 256, 0, s>>>(d, partial, nb);
  return 2;
}

int launch_philox_words(unsigned long long seed, unsigned long long step, unsigned long long cell0, long long n,
                        uint32_t* out, cudaStream_t s) {
  if (n <= 0) return 0;
  philox_words_kernel<<<cdiv(n, 256), 256, 0, s>>>(seed, step, cell0, n, reinterpret_cast<uint4*>(out));
  return 1;
}

}  // namespace avm
