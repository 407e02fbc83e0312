// avm_api.cu — the C ABI of include/avm.h: workspace carve-up, creation/validation, the step
// loop, state export in user order.  Host logic only enqueues work; the arithmetic of the hot
// path lives in avm_step.cu / avm_sort.cu.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include "avm_internal.cuh"

namespace avm {
int launch_hilbert_index(int m, long long n, const unsigned int* ix, const unsigned int* iy, unsigned int* out, cudaStream_t s);
int hilbert_bits(const Consts& k);
unsigned int hilbert_index_host(unsigned int x, unsigned int y, int m);
}

using namespace avm;

#ifndef AVM_FUSED_T1
#define AVM_FUSED_T1 1   // apply T1 flips in the prologue of the next force/move launch (two launches per step)
#endif

namespace {

thread_local std::string g_cuda_error;

#define AVM_CUDA(call)                                                                      \
  do {                                                                                      \
    cudaError_t e_ = (call);                                                                \
    if (e_ != cudaSuccess) {                                                                \
      g_cuda_error = std::string(#call) + ": " + cudaGetErrorString(e_);                    \
      return AVM_ECUDA;                                                                     \
    }                                                                                       \
  } while (0)

inline size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

inline int plane_stride(int V) { return (V + 63) & ~63; }

inline size_t dirty_words(size_t V) { return ((V + 31) / 32 + 31) & ~(size_t)31; }   // per bitmap

inline int t1_passes_of(const avm_params& p) { const int n = (p.flags & AVM_FLAG_T1_PASSES_MASK) >> AVM_FLAG_T1_PASSES_SHIFT; return n < 1 ? 1 : n; }

struct BufferSet {
  int *vn, *vc, *cvn, *vtag, *ctag;
  int4* cv;
  double* theta;
  rec_t* rec;
  CellPar* par;
};

struct Layout {
  size_t pos[2], vn[2], vc[2], cv[2], cvn[2], theta[2], rec[2], par[2], vtag[2], ctag[2];
  size_t img, msd_ref, img_stamp;
  size_t minkey, cand, ctr, dirty, estamp, ap, epart, key[2], val[2], hist, newidx_v, newidx_c, order_v, order_c;
  size_t total;
};

Layout make_layout(const avm_params& p) {
  Layout L;
  const size_t N = (size_t)p.n_cells, V = (size_t)p.n_vertices, S = (size_t)p.max_cell_vertices;
  const size_t Vs = (size_t)plane_stride(p.n_vertices);
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off += align_up(bytes); return o; };
  for (int i = 0; i < 2; ++i) L.pos[i] = take(16 * V);      // also staging for user-layout doubles: fp64 size in every build
  for (int i = 0; i < 2; ++i) {
    L.vn[i] = take(12 * Vs); L.vc[i] = take(12 * Vs); L.cv[i] = take(4 * N * S); L.cvn[i] = take(4 * N);
    L.theta[i] = take(8 * N); L.rec[i] = take(32 * N); L.par[i] = take(32 * N); L.vtag[i] = take(4 * V); L.ctag[i] = take(4 * N);
  }
  L.img = take(8 * V); L.msd_ref = take(16 * V); L.img_stamp = take(8 * V);
  L.minkey = take(8 * N);
  L.cand = take(sizeof(Cand) * (t1_passes_of(p) > 1 ? 5 : 3) * N);   // the step's list (3N = every edge) + two lists of N for repeated passes
  L.ctr = take(sizeof(Counters));
  L.dirty = take(4 * 2 * dirty_words(V));
  L.estamp = take(12 * Vs);
  L.ap = take(16 * N);
  L.epart = take(8 * 16 * (size_t)(cell_pass_grid(p.n_cells) > 512 ? cell_pass_grid(p.n_cells) : 512));   // block partials of the observables (up to 16 slots x the CTAs of the cell pass)
  for (int i = 0; i < 2; ++i) { L.key[i] = take(4 * V); L.val[i] = take(4 * V); }
  L.hist = take(4 * sort_hist_entries((int)V));
  L.newidx_v = take(4 * V); L.newidx_c = take(4 * N); L.order_v = take(4 * V); L.order_c = take(4 * N);
  L.total = off;
  return L;
}

bool params_ok(const avm_params* p) {
  if (!p) return false;
  if (p->n_cells < 4 || p->n_cells > (1 << 29)) return false;
  if (p->n_vertices != 2 * p->n_cells) return false;
  if (p->max_cell_vertices < 8 || p->max_cell_vertices > 32 || (p->max_cell_vertices & 3)) return false;
  { const int sch = p->flags & (AVM_FLAG_SCHEDULE_FUSED | AVM_FLAG_SCHEDULE_UNFUSED | AVM_FLAG_SCHEDULE_PERSISTENT); if (sch & (sch - 1)) return false; }   // at most one schedule flag
  if (!(p->Lx > 0.0) || !(p->Ly > 0.0) || !(p->dt >= 0.0) || !(p->l_c >= 0.0) || !(p->Dr >= 0.0)) return false;
  if (p->sort_every < 0) return false;
  return true;
}

}  // namespace

struct avm_sim {
  avm_params p;
  Consts k;
  cudaStream_t stream;
  char* ws;
  Layout L;
  pos_t* pos[2];
  BufferSet set[2];
  unsigned long long* minkey;
  Cand* cand;
  Counters* ctr;
  unsigned int* dirty;
  unsigned int* estamp;
  unsigned int* d_feedback;   // device view of h_feedback (or a word of the counters)
  int2* img;                  // MSD: image counts, user order
  double2* msd_ref;           // MSD: unwrapped reference positions, user order
  unsigned long long* img_stamp;   // MSD: step + 1 of the latest image-count update by a post-flip mover, user order
  bool tgt_custom, mod_custom;   // per-cell targets / moduli in force (Eq. 1); either one switches Consts::per_cell on
  unsigned int stamp;    // id of the latest repeated T1 pass (estamp entries equal to it were tested in that pass)
  int t1_passes;         // T1 passes per step (1 = north_star's rule; > 1 = repeat until none, NEXT-1)
  bool fused_ok;         // the two-launch schedule (T1 flips of a step ride in the next force/move launch) may be used
  bool fused_forced;     // ... and is used whatever the T1 load is (AVM_FLAG_SCHEDULE_FUSED)
  unsigned int* h_feedback;   // mapped host word (cudaHostAlloc): candidates of the latest completed step, written by
                              // every force/move launch; NULL if the allocation failed (the guess of avm_create is kept)
  unsigned int t1_guess;      // edges shorter than l_c at creation
  int persistent_grid;        // > 0: steps run inside one cooperative persistent launch with this many CTAs (launch-free stepping)
  double2* ap;
  double* epart;
  SortScratch sc;
  int cur_pos, cur_set;
  long long host_error;   // sticky bits raised by the host side (16: a persistent launch was refused), OR-ed into avm_stats.error
  unsigned long long step;
  long long n_sorts, launches;

  Dev dev() const {
    Dev d;
    d.pos = pos[cur_pos]; d.pos_next = pos[1 - cur_pos];
    const BufferSet& b = set[cur_set];
    d.vn = b.vn; d.vc = b.vc; d.cv = b.cv; d.cvn = b.cvn; d.theta = b.theta; d.rec = b.rec; d.par = b.par;
    d.vtag = b.vtag; d.ctag = b.ctag;
    d.minkey = minkey; d.cand = cand; d.ctr = ctr; d.dirty = dirty; d.estamp = estamp;
    d.feedback = d_feedback; d.img = img; d.msd_ref = msd_ref; d.img_stamp = img_stamp;
    return d;
  }
  Dev dev_alt() const {   // the other buffer set, target of a re-sort / staging area
    Dev d = dev();
    const BufferSet& b = set[1 - cur_set];
    d.pos = pos[1 - cur_pos]; d.pos_next = pos[cur_pos];
    d.vn = b.vn; d.vc = b.vc; d.cv = b.cv; d.cvn = b.cvn; d.theta = b.theta; d.rec = b.rec; d.par = b.par;
    d.vtag = b.vtag; d.ctag = b.ctag;
    return d;
  }
};

namespace {

// ---- creation-time kernels ---------------------------------------------------------------------
// user layout (staged in the alternate buffer set: vn/vc [V][3], cv [N][S] row-major) -> internal
// structure-of-arrays layout (vn/vc planes, cv int4 planes), tags, idle minimum keys
__global__ void import_kernel(const Dev d, const Consts k, const double* __restrict__ pos_u, const int* __restrict__ vn_u,
                              const int* __restrict__ vc_u, const int* __restrict__ cv_u) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < k.V) {
    d.vtag[i] = i;
    const double2 h = make_double2(pos_u[2 * i], pos_u[2 * i + 1]);
    const bool inside = h.x >= 0.0 && h.x < k.Lx && h.y >= 0.0 && h.y < k.Ly;
    if (!inside) atomicOr((unsigned long long*)&d.ctr->error, 4ull);
    pos_st(d.pos + i, inside ? h : make_double2(0.0, 0.0), k);
    d.img[i] = make_int2(0, 0);          // the mean-square displacement is measured from the initial state
    d.msd_ref[i] = pos_ld(d.pos + i, k);
#pragma unroll
    for (int s = 0; s < 3; ++s) { d.vn[s * k.Vs + i] = vn_u[3 * i + s]; d.vc[s * k.Vs + i] = vc_u[3 * i + s]; }
  }
  if (i < k.N) {
    d.ctag[i] = i;
    d.minkey[i] = ~0ull;
    int n = d.cvn[i];
    n = n < 0 ? 0 : (n > k.S ? k.S : n);
    for (int j = 0; j < k.S; ++j) row_entry(d.cv, k.N, i, j) = cv_u[(size_t)i * k.S + (j < n ? j : 0)];   // padding repeats entry 0
  }
}

// error bit 4: lists out of range or mutually inconsistent (slot convention, R12)
__global__ void validate_kernel(const Dev d, const Consts k) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  bool bad = false;
  if (i < k.N) {
    const int n = d.cvn[i];
    if (n < 3 || n > k.S) bad = true;
    else
      for (int j = 0; j < n; ++j) {
        const int v = row_entry(d.cv, k.N, i, j);
        if (v < 0 || v >= k.V) { bad = true; break; }
        const int c0 = d.vc[v], c1 = d.vc[k.Vs + v], c2 = d.vc[2 * k.Vs + v];
        if (c0 != i && c1 != i && c2 != i) bad = true;
      }
  }
  if (i < k.V) {
    for (int s = 0; s < 3 && !bad; ++s) {
      const int w = d.vn[s * k.Vs + i], c = d.vc[s * k.Vs + i], wn = d.vn[((s + 1) % 3) * k.Vs + i];
      if (w < 0 || w >= k.V || c < 0 || c >= k.N || w == i) { bad = true; break; }
      const int n = d.cvn[c];
      if (n < 3 || n > k.S) { bad = true; break; }
      int j = -1;
      for (int t = 0; t < n; ++t) if (row_entry(d.cv, k.N, c, t) == i) j = t;
      if (j < 0) { bad = true; break; }
      if (row_entry(d.cv, k.N, c, (j + 1) % n) != w || row_entry(d.cv, k.N, c, (j + n - 1) % n) != wn) bad = true;
    }
  }
  if (bad) atomicOr((unsigned long long*)&d.ctr->error, 4ull);
}

// ---- export in user order ------------------------------------------------------------------------
__global__ void export_vertices_kernel(const Dev d, const Consts k, double* pos, int* vn, int* vc) {
  const int v = blockIdx.x * blockDim.x + threadIdx.x;
  if (v >= k.V) return;
  const int t = d.vtag[v];
  if (pos) { const double2 h = pos_ld(d.pos + v, k); pos[2 * t] = h.x; pos[2 * t + 1] = h.y; }
  for (int s = 0; s < 3; ++s) {
    if (vn) vn[3 * t + s] = d.vtag[d.vn[s * k.Vs + v]];
    if (vc) vc[3 * t + s] = d.ctag[d.vc[s * k.Vs + v]];
  }
}
__global__ void export_cells_kernel(const Dev d, const Consts k, int* cvn, int* cv, double* theta) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= k.N) return;
  const int t = d.ctag[c];
  const int n = d.cvn[c];
  if (cvn) cvn[t] = n;
  if (theta) theta[t] = d.theta[c];
  if (cv)
    for (int j = 0; j < k.S; ++j) cv[(size_t)t * k.S + j] = j < n ? d.vtag[row_entry(d.cv, k.N, c, j)] : -1;
}
// which = 0: (A0_i, P0_i) <- (a, b); which = 1: (K_A,i, K_P,i) <- (a, b); user order in, internal order out.
// a == NULL restores the uniform pair; keep = 0 starts from the uniform values of avm_params.
__global__ void import_cell_params_kernel(const Dev d, const Consts k, const double* __restrict__ a, const double* __restrict__ b,
                                          const int which, const int keep) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= k.N) return;
  const int t = d.ctag[c];
  CellPar q;
  if (keep) q = d.par[c];
  else { q.A0 = k.A0; q.P0 = k.P0; q.KA = k.KA; q.KP = k.KP; }
  if (which == 0) { q.A0 = a ? a[t] : k.A0; q.P0 = a ? b[t] : k.P0; }
  else { q.KA = a ? a[t] : k.KA; q.KP = a ? b[t] : k.KP; }
  d.par[c] = q;
}
// overwrites the positions; the unwrapped positions and the MSD reference restart from them
__global__ void import_positions_kernel(const Dev d, const Consts k, const double* pos) {
  const int v = blockIdx.x * blockDim.x + threadIdx.x;
  if (v >= k.V) return;
  const int t = d.vtag[v];
  pos_st(d.pos + v, make_double2(pos[2 * t], pos[2 * t + 1]), k);
  d.msd_ref[t] = pos_ld(d.pos + v, k);
  d.img[t] = make_int2(0, 0);
}

inline int cdiv(long long a, int b) { return (int)((a + b - 1) / b); }

// the current unwrapped positions become the reference of the mean-square displacement
__global__ void msd_reset_kernel(const Dev d, const Consts k) {
  const int v = blockIdx.x * blockDim.x + threadIdx.x;
  if (v >= k.V) return;
  const int t = d.vtag[v];
  const double2 h = pos_ld(d.pos + v, k);
  const int2 im = d.img[t];
  d.msd_ref[t] = make_double2(h.x + (double)im.x * k.Lx, h.y + (double)im.y * k.Ly);
}

int do_sort(avm_sim* s) {
  const Dev a = s->dev(), b = s->dev_alt();
  s->launches += launch_t1_reset(a, s->k, s->stream);   // candidate lists hold pre-sort indices
  s->launches += launch_hilbert_sort(a, b, s->k, s->sc, s->stream);
  s->cur_pos = 1 - s->cur_pos;
  s->cur_set = 1 - s->cur_set;
  ++s->n_sorts;
  return AVM_OK;
}

// NEXT-1: the repeated T1 passes of the step just taken (s->step is still that step's index; the
// position buffers have been swapped already).  Lists alternate between ids 3 and 2.
int extra_t1_passes(avm_sim* s) {
  if (s->t1_passes <= 1) return 0;
  int n = 0;
  unsigned prev = (unsigned)(s->step & 1ull);
  for (int pass = 1; pass < s->t1_passes; ++pass) {
    const unsigned next = 2u + (unsigned)(pass & 1);
    if (++s->stamp == 0u) {               // wrapped: forget all stamps
      cudaMemsetAsync(s->estamp, 0, 12 * (size_t)s->k.Vs, s->stream);
      s->stamp = 1u;
    }
    n += launch_t1_extra_pass(s->dev(), s->k, prev, next, s->stamp, s->stream);
    prev = next;
  }
  return n + launch_t1_release(s->dev(), s->k, prev, s->stream);
}

int read_counters(avm_sim* s, Counters* out) {
  AVM_CUDA(cudaMemcpyAsync(out, s->ctr, sizeof(Counters), cudaMemcpyDeviceToHost, s->stream));
  AVM_CUDA(cudaStreamSynchronize(s->stream));
  return AVM_OK;
}

int create_common(const avm_params* params, const double* pos_xy, const int32_t* cvn, const int32_t* cv,
                  const int32_t* vn, const int32_t* vc, const double* theta, void* workspace,
                  size_t workspace_bytes, void* cuda_stream, avm_sim** out, bool host_inputs) {
  if (!out) return AVM_EINVAL;
  *out = nullptr;
  if (!params_ok(params) || !pos_xy || !cvn || !cv || !vn || !vc || !theta || !workspace) return AVM_EINVAL;
  const Layout L = make_layout(*params);
  if (workspace_bytes < L.total || ((uintptr_t)workspace & 255)) return AVM_EWORKSPACE;
  AVM_CUDA(cudaSetDevice(params->device));
  avm_sim* s = new (std::nothrow) avm_sim();
  if (!s) return AVM_ENOMEM;
  s->p = *params;
  s->stream = (cudaStream_t)cuda_stream;
  s->ws = (char*)workspace;
  s->L = L;
  const int N = params->n_cells, V = params->n_vertices, S = params->max_cell_vertices;
  Consts& k = s->k;
  k.N = N; k.V = V; k.S = S; k.Vs = plane_stride(V);
  k.Lx = params->Lx; k.Ly = params->Ly; k.hLx = 0.5 * params->Lx; k.hLy = 0.5 * params->Ly;
  k.KA = params->KA; k.KP = params->KP; k.KA2 = 2.0 * params->KA; k.KP2 = 2.0 * params->KP;
  k.A0 = params->A0; k.P0 = params->P0;
  k.v0_3 = params->v0 / 3.0; k.mu = params->mu; k.dt = params->dt;
  k.amp = sqrt(2.0 * params->Dr * params->dt);
  k.lc = params->l_c; k.lc2 = params->l_c * params->l_c;
  k.ux = params->Lx / 4294967296.0; k.uy = params->Ly / 4294967296.0; k.iux = 4294967296.0 / params->Lx; k.iuy = 4294967296.0 / params->Ly;
  k.seed = params->seed;
  k.per_cell = 0;
  k.cap_a = 3 * N;
  k.nw = (int)dirty_words((size_t)V);
  k.fm_grid = force_move_grid(V);
  for (int r = 0; r < 10; ++r) k.rkey[r] = philox_round_key(params->seed, r);
  char* w = s->ws;
  for (int i = 0; i < 2; ++i) {
    s->pos[i] = (pos_t*)(w + L.pos[i]);
    BufferSet& b = s->set[i];
    b.vn = (int*)(w + L.vn[i]); b.vc = (int*)(w + L.vc[i]); b.cv = (int4*)(w + L.cv[i]);
    b.cvn = (int*)(w + L.cvn[i]); b.theta = (double*)(w + L.theta[i]); b.rec = (rec_t*)(w + L.rec[i]); b.par = (CellPar*)(w + L.par[i]);
    b.vtag = (int*)(w + L.vtag[i]); b.ctag = (int*)(w + L.ctag[i]);
    s->sc.key[i] = (unsigned int*)(w + L.key[i]); s->sc.val[i] = (int*)(w + L.val[i]);
  }
  s->img = (int2*)(w + L.img); s->msd_ref = (double2*)(w + L.msd_ref); s->img_stamp = (unsigned long long*)(w + L.img_stamp);
  s->tgt_custom = s->mod_custom = false;
  s->minkey = (unsigned long long*)(w + L.minkey);
  s->cand = (Cand*)(w + L.cand);
  s->ctr = (Counters*)(w + L.ctr);
  s->dirty = (unsigned int*)(w + L.dirty);
  s->estamp = (unsigned int*)(w + L.estamp);
  s->stamp = 0;
  s->ap = (double2*)(w + L.ap);
  s->epart = (double*)(w + L.epart);
  s->sc.hist = (unsigned int*)(w + L.hist);
  s->sc.newidx_v = (int*)(w + L.newidx_v); s->sc.newidx_c = (int*)(w + L.newidx_c);
  s->sc.order_v = (int*)(w + L.order_v); s->sc.order_c = (int*)(w + L.order_c);
  s->cur_pos = 0; s->cur_set = 0;
  s->step = params->step0;
  s->n_sorts = 0; s->launches = 0; s->host_error = 0;
  // Two-launch schedule (flips inside the next force/move launch) pays when the sweep is longer
  // than the flippers' chain of dependent loads (~15 us): from about a million vertices; and for
  // tiny systems, which flip rarely and are bound by the number of launches.  In between the plain
  // three-launch schedule is faster.  AVM_FLAG_SCHEDULE_FUSED / _UNFUSED override (both give the same bits).
  s->t1_passes = t1_passes_of(*params);
  s->fused_forced = (params->flags & AVM_FLAG_SCHEDULE_FUSED) != 0;
  s->fused_ok = s->t1_passes == 1 && AVM_FUSED_T1 && (V >= (1 << 20) || V <= 2048 || s->fused_forced) &&
                !(params->flags & AVM_FLAG_SCHEDULE_UNFUSED);
  k.flag_dirty = 0; k.clear_dirty = 0;
  // Launch-free stepping: ONE launch per avm_step call (or per stretch between re-sorts), bit-identical to the other
  // schedules.  Default up to 8192 vertices: one CTA up to 512 vertices (barriers are
  // __syncthreads, cached loads: 1.97 us/step at configs[0] against 4.8 with two launches per step), one thread-block
  // CLUSTER of up to 16 CTAs with the hardware cluster barrier beyond (8.1 against 9.8 us at configs[1]).  Above that a
  // step is a chain of ~8 dependent L2 round trips plus barriers either way and one launch per kernel is faster
  // (15.0 against 20.6 us at configs[2]); AVM_FLAG_SCHEDULE_PERSISTENT still selects it for any size (a cooperative
  // grid with an arrival-counter barrier).
  s->persistent_grid = 0;
  {
    const bool forced = (params->flags & AVM_FLAG_SCHEDULE_PERSISTENT) != 0;
    const bool other = (params->flags & (AVM_FLAG_SCHEDULE_FUSED | AVM_FLAG_SCHEDULE_UNFUSED)) != 0;
    if (s->t1_passes == 1 && !other && (forced || V <= 8192)) s->persistent_grid = persistent_grid(V, false);
  }
  s->h_feedback = nullptr;
  s->d_feedback = &s->ctr->feedback_sink;
  s->t1_guess = 0;
  if (s->fused_ok && !s->fused_forced) {
    void* h = nullptr;
    void* dptr = nullptr;
    if (cudaHostAlloc(&h, 64, cudaHostAllocMapped) == cudaSuccess && cudaHostGetDevicePointer(&dptr, h, 0) == cudaSuccess) {
      s->h_feedback = (unsigned int*)h;
      s->d_feedback = (unsigned int*)dptr;
    } else {
      if (h) cudaFreeHost(h);
      cudaGetLastError();
    }
  }

  cudaStream_t st = s->stream;
  const cudaMemcpyKind kind = host_inputs ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice;
  const BufferSet& b = s->set[0];
  const BufferSet& stage = s->set[1];   // user-layout staging for the import kernel
  auto fail = [&](int code) { if (s->h_feedback) cudaFreeHost(s->h_feedback); delete s; return code; };
#define AVM_CUDA_F(call)                                                                    \
  do {                                                                                      \
    cudaError_t e_ = (call);                                                                \
    if (e_ != cudaSuccess) {                                                                \
      g_cuda_error = std::string(#call) + ": " + cudaGetErrorString(e_);                    \
      return fail(AVM_ECUDA);                                                               \
    }                                                                                       \
  } while (0)
  AVM_CUDA_F(cudaMemcpyAsync(s->pos[1], pos_xy, 16 * (size_t)V, kind, st));    // user-layout doubles, packed by the import kernel
  AVM_CUDA_F(cudaMemcpyAsync(stage.vn, vn, 12 * (size_t)V, kind, st));
  AVM_CUDA_F(cudaMemcpyAsync(stage.vc, vc, 12 * (size_t)V, kind, st));
  AVM_CUDA_F(cudaMemcpyAsync(stage.cv, cv, 4 * (size_t)N * S, kind, st));
  AVM_CUDA_F(cudaMemcpyAsync(b.cvn, cvn, 4 * (size_t)N, kind, st));
  AVM_CUDA_F(cudaMemcpyAsync(b.theta, theta, 8 * (size_t)N, kind, st));
  AVM_CUDA_F(cudaMemsetAsync(s->ctr, 0, sizeof(Counters), st));
  AVM_CUDA_F(cudaMemsetAsync(s->dirty, 0, 4 * 2 * (size_t)k.nw, st));
  AVM_CUDA_F(cudaMemsetAsync(s->estamp, 0, 12 * (size_t)k.Vs, st));
  AVM_CUDA_F(cudaMemsetAsync(s->img_stamp, 0, 8 * (size_t)V, st));     // 0 = never (a stamp is step + 1 >= 1)
  const Dev d = s->dev();
  import_kernel<<<cdiv(V, 256), 256, 0, st>>>(d, k, (const double*)s->pos[1], stage.vn, stage.vc, (const int*)stage.cv);
  validate_kernel<<<cdiv(V, 256), 256, 0, st>>>(d, k);
  s->launches += 2;
  s->launches += launch_count_short_edges(d, k, st);      // first guess of the T1 load (into ctr->n_win)
  Counters c;
  AVM_CUDA_F(cudaMemcpyAsync(&c, s->ctr, sizeof(Counters), cudaMemcpyDeviceToHost, st));
  AVM_CUDA_F(cudaStreamSynchronize(st));
  AVM_CUDA_F(cudaGetLastError());
  if (c.error & 4) return fail(AVM_EINCONSISTENT);
  s->t1_guess = c.n_win;
  if (s->h_feedback) *s->h_feedback = s->t1_guess;
  // the device rewrites the host word only when the load crosses the schedule threshold: both sides start from the guess
  AVM_CUDA_F(cudaMemcpyAsync(&s->ctr->fb_last, &s->t1_guess, sizeof(unsigned int), cudaMemcpyHostToDevice, st));
  s->launches += launch_refresh_cells(d, k, st);
  if (params->flags & AVM_FLAG_SORT_AT_CREATE) do_sort(s);
  AVM_CUDA_F(cudaGetLastError());
#undef AVM_CUDA_F
  *out = s;
  return AVM_OK;
}

int get_state_common(avm_sim* s, double* pos_xy, int32_t* cvn, int32_t* cv, int32_t* vn, int32_t* vc,
                     double* theta, avm_stats* stats, bool host_outputs) {
  if (!s) return AVM_EINVAL;
  const Consts& k = s->k;
  const Dev d = s->dev();
  cudaStream_t st = s->stream;
  if (!host_outputs) {
    if (pos_xy || vn || vc) { export_vertices_kernel<<<cdiv(k.V, 256), 256, 0, st>>>(d, k, pos_xy, vn, vc); ++s->launches; }
    if (cvn || cv || theta) { export_cells_kernel<<<cdiv(k.N, 256), 256, 0, st>>>(d, k, cvn, cv, theta); ++s->launches; }
  } else {
    // stage in the idle buffers (ping-pong partner of pos, alternate buffer set), then copy out
    const Dev a = s->dev_alt();
    double* spos = (double*)a.pos;
    if (pos_xy || vn || vc) {
      export_vertices_kernel<<<cdiv(k.V, 256), 256, 0, st>>>(d, k, pos_xy ? spos : nullptr, vn ? a.vn : nullptr, vc ? a.vc : nullptr);
      ++s->launches;
    }
    if (cvn || cv || theta) {
      export_cells_kernel<<<cdiv(k.N, 256), 256, 0, st>>>(d, k, cvn ? a.cvn : nullptr, cv ? (int*)a.cv : nullptr, theta ? a.theta : nullptr);
      ++s->launches;
    }
    if (pos_xy) AVM_CUDA(cudaMemcpyAsync(pos_xy, spos, 16 * (size_t)k.V, cudaMemcpyDeviceToHost, st));
    if (vn) AVM_CUDA(cudaMemcpyAsync(vn, a.vn, 12 * (size_t)k.V, cudaMemcpyDeviceToHost, st));
    if (vc) AVM_CUDA(cudaMemcpyAsync(vc, a.vc, 12 * (size_t)k.V, cudaMemcpyDeviceToHost, st));
    if (cvn) AVM_CUDA(cudaMemcpyAsync(cvn, a.cvn, 4 * (size_t)k.N, cudaMemcpyDeviceToHost, st));
    if (cv) AVM_CUDA(cudaMemcpyAsync(cv, a.cv, 4 * (size_t)k.N * k.S, cudaMemcpyDeviceToHost, st));
    if (theta) AVM_CUDA(cudaMemcpyAsync(theta, a.theta, 8 * (size_t)k.N, cudaMemcpyDeviceToHost, st));
  }
  if (stats) {
    Counters c;
    int rc = read_counters(s, &c);
    if (rc) return rc;
    stats->step = (int64_t)s->step;
    stats->t1_short = c.t1_short; stats->t1_candidates = c.t1_candidates; stats->t1_flips = c.t1_flips;
    stats->t1_blocked = c.t1_blocked; stats->overflow_rejects = c.overflow_rejects; stats->error = c.error | s->host_error;
    stats->n_sorts = s->n_sorts; stats->kernel_launches = s->launches;
  } else if (host_outputs) {
    AVM_CUDA(cudaStreamSynchronize(st));
  }
  AVM_CUDA(cudaGetLastError());
  return AVM_OK;
}

}  // namespace

// ===============================================================================================
extern "C" {

size_t avm_workspace_bytes(const avm_params* params) {
  if (!params_ok(params)) return 0;
  return make_layout(*params).total;
}

int avm_create(const avm_params* params, const double* pos_xy, const int32_t* cell_vertex_num,
               const int32_t* cell_vertices, const int32_t* vertex_neighbors,
               const int32_t* vertex_cell_neighbors, const double* theta, void* workspace,
               size_t workspace_bytes, void* cuda_stream, avm_sim** out) {
  return create_common(params, pos_xy, cell_vertex_num, cell_vertices, vertex_neighbors, vertex_cell_neighbors,
                       theta, workspace, workspace_bytes, cuda_stream, out, false);
}

int avm_create_host(const avm_params* params, const double* pos_xy, const int32_t* cell_vertex_num,
                    const int32_t* cell_vertices, const int32_t* vertex_neighbors,
                    const int32_t* vertex_cell_neighbors, const double* theta, void* workspace,
                    size_t workspace_bytes, void* cuda_stream, avm_sim** out) {
  return create_common(params, pos_xy, cell_vertex_num, cell_vertices, vertex_neighbors, vertex_cell_neighbors,
                       theta, workspace, workspace_bytes, cuda_stream, out, true);
}

// Schedule of one step.  Leaving the flips of a step pending (they then ride
// in the next force/move launch: two launches per step) pays while there are few candidates: a few
// dedicated warps handle them in the shadow of the sweep.  With many candidates the stand-alone T1
// kernel is faster (more registers, quiet SMs).  The load is known from the count every force/move
// launch reports through a mapped host word (read here without synchronising; it lags the device by
// however far the host runs ahead, which is fine for a slowly varying load), before that from the
// number of short edges at creation.  Both schedules give the same bits.
static bool leave_flips_pending(const avm_sim* s, bool last_of_call) {
  if (!s->fused_ok || last_of_call) return false;   // the last step of a call is completed inside the call
  if (s->p.sort_every > 0 && (s->step + 1 - s->p.step0) % (unsigned long long)s->p.sort_every == 0) return false;   // so is the step before a re-sort
  if (s->fused_forced) return true;
  const unsigned load = s->h_feedback ? *(volatile unsigned int*)s->h_feedback : s->t1_guess;
  return load <= AVM_FUSED_MAX_CANDIDATES;
}

int avm_step(avm_sim* s, int64_t n_steps) {
  if (!s || n_steps < 0) return AVM_EINVAL;
  if (s->persistent_grid > 0) {
    int64_t done = 0;
    while (done < n_steps) {
      int64_t chunk = n_steps - done < 65536 ? n_steps - done : 65536;
      if (s->p.sort_every > 0) {                       // stop at the next re-sort
        const int64_t to_sort = (int64_t)s->p.sort_every - (int64_t)((s->step - s->p.step0) % (unsigned long long)s->p.sort_every);
        if (to_sort < chunk) chunk = to_sort;
      }
      const int grid = s->k.per_cell ? persistent_grid(s->k.V, true) : s->persistent_grid;
      const int n = grid > 0 ? launch_persistent_steps(s->dev(), s->k, s->step, (int)chunk, grid, s->stream) : -1;
      if (n < 0) { s->persistent_grid = 0; s->host_error |= 16; break; }    // refused: go on with one launch per kernel, and say so (avm_stats.error)
      s->launches += n;
      if (chunk & 1) s->cur_pos = 1 - s->cur_pos;
      s->step += (unsigned long long)chunk;
      done += chunk;
      if (s->p.sort_every > 0 && (s->step - s->p.step0) % (unsigned long long)s->p.sort_every == 0) do_sort(s);
    }
    if (done == n_steps) { AVM_CUDA(cudaPeekAtLastError()); return AVM_OK; }
    n_steps -= done;
  }
  bool pending = false;     // the previous step of this call left its flips pending
  for (int64_t i = 0; i < n_steps; ++i) {
    const bool leave = leave_flips_pending(s, i == n_steps - 1);
    s->launches += launch_step(s->dev(), s->k, s->step, s->stream, nullptr, pending, leave);
    pending = leave;
    s->cur_pos = 1 - s->cur_pos;
    s->launches += extra_t1_passes(s);
    ++s->step;
    if (s->p.sort_every > 0 && (s->step - s->p.step0) % (unsigned long long)s->p.sort_every == 0) do_sort(s);
  }
  AVM_CUDA(cudaPeekAtLastError());
  return AVM_OK;
}


int avm_step_profile(avm_sim* s, int64_t n_steps, double* ms_per_kernel) {
  if (!s || n_steps < 0 || !ms_per_kernel) return AVM_EINVAL;
  cudaEvent_t ev[AVM_K_COUNT + 1];
  for (int i = 0; i <= AVM_K_COUNT; ++i) AVM_CUDA(cudaEventCreate(&ev[i]));
  for (int i = 0; i < AVM_K_COUNT; ++i) ms_per_kernel[i] = 0.0;
  // One launch per kernel, with avm_step's choice between two and three launches per step; the events serialise
  // the launches.  The launch-free persistent kernel (avm_step's default up to 8192 vertices) has no kernel
  // boundaries to bracket and is never taken here, so for such systems these times describe the launched schedule.
  bool pending = false;
  for (int64_t i = 0; i < n_steps; ++i) {
    const bool leave = leave_flips_pending(s, i == n_steps - 1);
    s->launches += launch_step(s->dev(), s->k, s->step, s->stream, ev, pending, leave);
    pending = leave;
    s->cur_pos = 1 - s->cur_pos;
    s->launches += extra_t1_passes(s);                  // outside the per-kernel slots
    ++s->step;
    AVM_CUDA(cudaEventSynchronize(ev[AVM_K_COUNT]));
    for (int j = 0; j < AVM_K_COUNT; ++j) {
      float ms = 0.f;
      AVM_CUDA(cudaEventElapsedTime(&ms, ev[j], ev[j + 1]));
      if (!(leave && j == AVM_K_T1_FLIP)) ms_per_kernel[j] += ms;   // two-launch step: nothing ran in that slot
    }
    if (s->p.sort_every > 0 && (s->step - s->p.step0) % (unsigned long long)s->p.sort_every == 0) do_sort(s);
  }
  for (int i = 0; i <= AVM_K_COUNT; ++i) cudaEventDestroy(ev[i]);
  AVM_CUDA(cudaGetLastError());
  return AVM_OK;
}

int avm_compute_forces(avm_sim* s, double* force_xy, double* area_perim) {
  if (!s) return AVM_EINVAL;
  s->launches += launch_compute_forces(s->dev(), s->k, s->ap, force_xy, area_perim, s->stream);
  AVM_CUDA(cudaPeekAtLastError());
  return AVM_OK;
}

int avm_compute_forces_host(avm_sim* s, double* force_xy, double* area_perim) {
  if (!s) return AVM_EINVAL;
  const Dev a = s->dev_alt();
  double* sf = (double*)a.pos;      // idle ping-pong partner
  double* sap = (double*)a.rec;     // idle alternate record buffer (32N bytes >= 16N)
  s->launches += launch_compute_forces(s->dev(), s->k, s->ap, force_xy ? sf : nullptr, area_perim ? sap : nullptr, s->stream);
  if (force_xy) AVM_CUDA(cudaMemcpyAsync(force_xy, sf, 16 * (size_t)s->k.V, cudaMemcpyDeviceToHost, s->stream));
  if (area_perim) AVM_CUDA(cudaMemcpyAsync(area_perim, sap, 16 * (size_t)s->k.N, cudaMemcpyDeviceToHost, s->stream));
  AVM_CUDA(cudaStreamSynchronize(s->stream));
  AVM_CUDA(cudaGetLastError());
  return AVM_OK;
}

int avm_energy(avm_sim* s, double* energy) {
  if (!s || !energy) return AVM_EINVAL;
  s->launches += launch_energy(s->dev(), s->k, s->epart, s->stream);
  Counters c;
  int rc = read_counters(s, &c);
  if (rc) return rc;
  *energy = c.obs[0];
  return AVM_OK;
}

static int fill_observables(avm_sim* s, avm_observables* out);

int avm_observe(avm_sim* s, avm_observables* out) {
  if (!s || !out) return AVM_EINVAL;
  s->launches += launch_energy(s->dev(), s->k, s->epart, s->stream);
  return fill_observables(s, out);
}

int avm_step_observe(avm_sim* s, int64_t n_steps, avm_observables* out) {
  if (!s || !out || n_steps < 1) return AVM_EINVAL;
  int rc = avm_step(s, n_steps - 1);            // whole steps: the last one of that call is completed inside it
  if (rc) return rc;
  s->launches += launch_step(s->dev(), s->k, s->step, s->stream, nullptr, false, false, s->epart);
  s->cur_pos = 1 - s->cur_pos;
  s->launches += extra_t1_passes(s);
  ++s->step;
  if (s->p.sort_every > 0 && (s->step - s->p.step0) % (unsigned long long)s->p.sort_every == 0) do_sort(s);
  return fill_observables(s, out);
}

static int fill_observables(avm_sim* s, avm_observables* out) {
  Counters c;
  int rc = read_counters(s, &c);
  if (rc) return rc;
  const double N = (double)s->k.N;
  out->energy = c.obs[0];
  out->sum_area = c.obs[1];
  out->sum_perimeter = c.obs[2];
  out->n_nonpositive_area = (int64_t)c.obs[4];
  const double npos = N - c.obs[4];
  out->mean_shape_index = npos > 0.0 ? c.obs[3] / npos : 0.0;
  out->area_variance = c.obs[5] / N - (c.obs[1] / N) * (c.obs[1] / N);
  out->area_min = c.obs[6];
  out->area_max = c.obs[7];
  out->msd = c.obs[8] / (double)s->k.V;
  out->step = (int64_t)s->step;
  out->t1_flips = c.t1_flips;
  return AVM_OK;
}

int avm_get_state(avm_sim* s, double* pos_xy, int32_t* cell_vertex_num, int32_t* cell_vertices,
                  int32_t* vertex_neighbors, int32_t* vertex_cell_neighbors, double* theta, avm_stats* stats) {
  return get_state_common(s, pos_xy, cell_vertex_num, cell_vertices, vertex_neighbors, vertex_cell_neighbors, theta, stats, false);
}

int avm_get_state_host(avm_sim* s, double* pos_xy, int32_t* cell_vertex_num, int32_t* cell_vertices,
                       int32_t* vertex_neighbors, int32_t* vertex_cell_neighbors, double* theta, avm_stats* stats) {
  return get_state_common(s, pos_xy, cell_vertex_num, cell_vertices, vertex_neighbors, vertex_cell_neighbors, theta, stats, true);
}

int avm_debug_t1(avm_sim* s, int32_t* cand_pairs, int64_t* n_cand, int32_t* winner_pairs, int64_t* n_win, int64_t capacity) {
  if (!s || !n_cand || !n_win || capacity < 0) return AVM_EINVAL;
  const Dev a = s->dev_alt();
  // staging in idle alternate buffers: cv (4*N*S bytes) and rec (32*N bytes) hold >= 3N/4N pairs
  int* sc = (int*)a.cv;
  int* sw = (int*)a.rec;
  const long long cap_c = (long long)s->k.N * s->k.S / 2, cap_w = (long long)s->k.N * 4;
  const long long cc = capacity < cap_c ? capacity : cap_c, cw = capacity < cap_w ? capacity : cap_w;
  s->launches += launch_t1_debug(s->dev(), s->k, cand_pairs ? sc : nullptr, winner_pairs ? sw : nullptr, cc < cw ? cc : cw, s->stream);
  Counters c;
  int rc = read_counters(s, &c);
  if (rc) return rc;
  *n_cand = c.n_cand[0]; *n_win = c.n_win;
  const long long lim = cc < cw ? cc : cw;
  const long long ncopy = (long long)c.n_cand[0] < lim ? (long long)c.n_cand[0] : lim;
  const long long wcopy = (long long)c.n_win < lim ? (long long)c.n_win : lim;
  if (cand_pairs && ncopy) AVM_CUDA(cudaMemcpyAsync(cand_pairs, sc, 8 * (size_t)ncopy, cudaMemcpyDeviceToHost, s->stream));
  if (winner_pairs && wcopy) AVM_CUDA(cudaMemcpyAsync(winner_pairs, sw, 8 * (size_t)wcopy, cudaMemcpyDeviceToHost, s->stream));
  s->launches += launch_t1_reset(s->dev(), s->k, s->stream);
  AVM_CUDA(cudaStreamSynchronize(s->stream));
  return AVM_OK;
}

int avm_t1_pass(avm_sim* s) {
  if (!s) return AVM_EINVAL;
  s->launches += launch_t1_pass_only(s->dev(), s->k, s->stream);
  AVM_CUDA(cudaPeekAtLastError());
  return AVM_OK;
}

int avm_set_positions(avm_sim* s, const double* pos_xy) {
  if (!s || !pos_xy) return AVM_EINVAL;
  const Dev d = s->dev();
  import_positions_kernel<<<cdiv(s->k.V, 256), 256, 0, s->stream>>>(d, s->k, pos_xy);
  ++s->launches;
  s->launches += launch_refresh_cells(d, s->k, s->stream);
  AVM_CUDA(cudaPeekAtLastError());
  return AVM_OK;
}

static int set_cell_params(avm_sim* s, const double* a, const double* b, int which) {
  if (!s || ((a == nullptr) != (b == nullptr))) return AVM_EINVAL;
  const int keep = s->k.per_cell;
  (which == 0 ? s->tgt_custom : s->mod_custom) = a != nullptr;
  const Dev d = s->dev();
  import_cell_params_kernel<<<cdiv(s->k.N, 256), 256, 0, s->stream>>>(d, s->k, a, b, which, keep);
  ++s->launches;
  s->k.per_cell = (s->tgt_custom || s->mod_custom) ? 1 : 0;
  s->launches += launch_refresh_cells(s->dev(), s->k, s->stream);   // the cached records hold 2 K_A,i (A - A0_i), 2 K_P,i (P - P0_i)
  AVM_CUDA(cudaPeekAtLastError());
  return AVM_OK;
}

int avm_set_cell_targets(avm_sim* s, const double* area0, const double* perimeter0) { return set_cell_params(s, area0, perimeter0, 0); }

int avm_set_cell_moduli(avm_sim* s, const double* KA, const double* KP) { return set_cell_params(s, KA, KP, 1); }

int avm_msd_reset(avm_sim* s) {
  if (!s) return AVM_EINVAL;
  msd_reset_kernel<<<cdiv(s->k.V, 256), 256, 0, s->stream>>>(s->dev(), s->k);
  ++s->launches;
  AVM_CUDA(cudaPeekAtLastError());
  return AVM_OK;
}

// ---- SPV on a fixed triangulation (avm_spv.cu) ----
static int spv_refresh(avm_sim* s, const double* cell_xy, double* voronoi_xy) {
  s->launches += launch_spv_voronoi(s->dev(), s->k, cell_xy, voronoi_xy, s->stream);
  s->launches += launch_refresh_cells(s->dev(), s->k, s->stream);
  return AVM_OK;
}

int avm_spv_geometry(avm_sim* s, const double* cell_xy, double* voronoi_xy, double* area_perim) {
  if (!s || !cell_xy) return AVM_EINVAL;
  spv_refresh(s, cell_xy, voronoi_xy);
  if (area_perim) s->launches += launch_compute_forces(s->dev(), s->k, s->ap, nullptr, area_perim, s->stream);
  AVM_CUDA(cudaPeekAtLastError());
  return AVM_OK;
}

int avm_spv_forces(avm_sim* s, const double* cell_xy, double* force_xy, double* force_sets) {
  if (!s || !cell_xy) return AVM_EINVAL;
  spv_refresh(s, cell_xy, nullptr);
  const Dev d = s->dev();
  s->launches += launch_spv_forces(d, s->k, cell_xy, (double2*)d.pos_next, s->ap, force_xy, force_sets, s->stream);
  AVM_CUDA(cudaPeekAtLastError());
  return AVM_OK;
}

static int spv_read_counts(avm_sim* s, int64_t* n_failed, bool with_first) {
  unsigned long long c[2];
  AVM_CUDA(cudaMemcpyAsync(c, s->ctr->spv, sizeof(c), cudaMemcpyDeviceToHost, s->stream));
  AVM_CUDA(cudaStreamSynchronize(s->stream));
  n_failed[0] = (int64_t)c[0];
  if (with_first) n_failed[1] = c[1] == ~0ull ? -1 : (int64_t)c[1];
  return AVM_OK;
}

int avm_spv_test_triangulation(avm_sim* s, const double* cell_xy, int64_t* n_failed, int32_t* cell_flags) {
  if (!s || !cell_xy || !n_failed) return AVM_EINVAL;
  AVM_CUDA(cudaMemsetAsync(s->ctr->spv, 0, sizeof(unsigned long long), s->stream));
  AVM_CUDA(cudaMemsetAsync(s->ctr->spv + 1, 0xff, sizeof(unsigned long long), s->stream));
  if (cell_flags) AVM_CUDA(cudaMemsetAsync(cell_flags, 0, sizeof(int32_t) * (size_t)s->k.N, s->stream));
  s->launches += launch_spv_test(s->dev(), s->k, cell_xy, s->ctr->spv, cell_flags, 0ull, s->stream);
  return spv_read_counts(s, n_failed, false);
}

int avm_spv_step(avm_sim* s, double* cell_xy, int64_t n_steps, int64_t* n_failed, int32_t* cell_flags) {
  if (!s || !cell_xy || !n_failed || n_steps < 0) return AVM_EINVAL;
  AVM_CUDA(cudaMemsetAsync(s->ctr->spv, 0, sizeof(unsigned long long), s->stream));
  AVM_CUDA(cudaMemsetAsync(s->ctr->spv + 1, 0xff, sizeof(unsigned long long), s->stream));
  for (int64_t i = 0; i < n_steps; ++i) {
    spv_refresh(s, cell_xy, nullptr);
    const Dev d = s->dev();
    s->launches += launch_spv_forces(d, s->k, cell_xy, (double2*)d.pos_next, s->ap, nullptr, nullptr, s->stream);   // :86-88
    s->launches += launch_spv_move(d, s->k, cell_xy, s->ap, s->p.v0, s->step, s->stream);                            // Eq. 3, :92
    ++s->step;
    AVM_CUDA(cudaMemsetAsync(s->ctr->spv, 0, sizeof(unsigned long long), s->stream));
    if (cell_flags) AVM_CUDA(cudaMemsetAsync(cell_flags, 0, sizeof(int32_t) * (size_t)s->k.N, s->stream));
    s->launches += launch_spv_test(d, s->k, cell_xy, s->ctr->spv, cell_flags, (unsigned long long)i, s->stream);      // :94
  }
  spv_refresh(s, cell_xy, nullptr);      // the simulation's vertex positions and records describe the final cells
  return spv_read_counts(s, n_failed, true);
}

int avm_resort(avm_sim* s) {
  if (!s) return AVM_EINVAL;
  do_sort(s);
  AVM_CUDA(cudaPeekAtLastError());
  return AVM_OK;
}

int avm_philox_words(avm_sim* s, uint64_t seed, uint64_t step, uint64_t cell0, int64_t n, uint32_t* out_words) {
  if (!s || !out_words || n < 0) return AVM_EINVAL;
  s->launches += launch_philox_words(seed, step, cell0, n, out_words, s->stream);
  AVM_CUDA(cudaPeekAtLastError());
  return AVM_OK;
}

int avm_hilbert_index(avm_sim* s, int32_t m, int64_t n, const uint32_t* ix, const uint32_t* iy, uint32_t* out) {
  if (!s || m < 1 || m > 16 || n < 0 || !ix || !iy || !out) return AVM_EINVAL;
  s->launches += launch_hilbert_index(m, n, ix, iy, out, s->stream);
  AVM_CUDA(cudaPeekAtLastError());
  return AVM_OK;
}

uint32_t avm_hilbert_index_host(int32_t m, uint32_t ix, uint32_t iy) {
  if (m < 1 || m > 16) return 0;
  return hilbert_index_host(ix, iy, m);
}

void avm_destroy(avm_sim* s) {
  if (!s) return;
  if (s->h_feedback) cudaFreeHost(s->h_feedback);
  delete s;
}

const char* avm_strerror(int code) {
  switch (code) {
    case AVM_OK: return "ok";
    case AVM_EINVAL: return "invalid argument (NULL pointer, V != 2N, bad stride or parameter)";
    case AVM_EWORKSPACE: return "workspace too small or not 256-byte aligned";
    case AVM_EINCONSISTENT: return "topology lists are out of range or inconsistent with each other";
    case AVM_ECUDA: return "CUDA error (see avm_last_cuda_error)";
    case AVM_ENOMEM: return "out of host memory";
    case AVM_ETOOLARGE: return "more cells than avm_forces_static's fixed scratch array holds (AVM_FORCES_STATIC_MAX_CELLS)";
    default: return "unknown error";
  }
}

const char* avm_last_cuda_error(void) { return g_cuda_error.c_str(); }

const char* avm_precision(void) { return AVM_MIXED ? "mixed" : "f64"; }

}  // extern "C"

// for the entry points that live in other files (avm_forces_static.cu)
namespace avm {
void note_cuda_error(const char* call, cudaError_t e) { g_cuda_error = std::string(call) + ": " + cudaGetErrorString(e); }
}
