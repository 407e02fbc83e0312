// avm_sort.cu — row H of the hot path: periodic Hilbert-curve re-ordering of cells and vertices
// (§II.B: "uses a Hilbert-curve-based spatial sorting scheme ... finds the location
// on the curve closest to each cell, and sorts cells based on the order in which they occur";
// effect on the GPU: PAPER.md:116, :126).  DESIGN.md R18.
//
// Everything is hand-written: Hilbert keys, a stable least-significant-digit radix sort
// (8 bits per pass, warp-private digit counters so the scatter is stable and deterministic),
// the permutation of every array and the re-indexing of every stored index.  Tags (user
// indices) travel with the data, so user-visible order, Philox keys and T1 priorities never
// change.  Runs every `sort_every` steps: off the per-step path.
#include "avm_internal.cuh"

namespace avm {

static constexpr int kSeg = 2048;       // elements per warp segment
static constexpr int kWarpsPerBlock = 8;

// Hilbert index of grid cell (x, y) on a 2^m x 2^m grid: walk from the coarsest quadrant down,
// accumulating quadrant ranks and applying the quadrant's reflection/transpose to the remainder.
__device__ __host__ __forceinline__ unsigned int hilbert_index(unsigned int x, unsigned int y, int m) {
  unsigned int d = 0;
  for (int b = m - 1; b >= 0; --b) {
    const unsigned int s = 1u << b;
    const unsigned int rx = (x >> b) & 1u, ry = (y >> b) & 1u;
    d += s * s * ((3u * rx) ^ ry);
    // keep only the bits below b, reflected/transposed into the sub-quadrant's frame
    x &= s - 1u; y &= s - 1u;
    if (ry == 0u) {
      if (rx == 1u) { x = (s - 1u) - x; y = (s - 1u) - y; }
      const unsigned int t = x; x = y; y = t;
    }
  }
  return d;
}

__device__ __forceinline__ unsigned int key_of_position(double x, double y, const Consts& k, int m) {
  const unsigned int g = 1u << m;
  int ix = (int)floor(x / k.Lx * (double)g), iy = (int)floor(y / k.Ly * (double)g);
  ix = ix < 0 ? 0 : (ix >= (int)g ? (int)g - 1 : ix);
  iy = iy < 0 ? 0 : (iy >= (int)g ? (int)g - 1 : iy);
  return hilbert_index((unsigned int)ix, (unsigned int)iy, m);
}

// keys are laid out in TAG order (slot t belongs to the vertex whose tag is t) so that the stable
// sort breaks ties by tag whatever the current order is; the payload is the current index.
__global__ void vertex_keys_kernel(const Dev d, const Consts k, int m, unsigned int* __restrict__ key, int* __restrict__ val) {
  const int v = blockIdx.x * blockDim.x + threadIdx.x;
  if (v >= k.V) return;
  const double2 h = d.pos[v];
  const int t = d.vtag[v];
  key[t] = key_of_position(h.x, h.y, k, m);
  val[t] = v;
}

__global__ void cell_keys_kernel(const Dev d, const Consts k, int m, unsigned int* __restrict__ key, int* __restrict__ val) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= k.N) return;
  const int n = d.cvn[c];
  const double2 h0 = d.pos[row_entry(d.cv, k.N, c, 0)];
  double sx = 0.0, sy = 0.0;
  for (int j = 1; j < n; ++j) {
    const double2 hj = d.pos[row_entry(d.cv, k.N, c, j)];
    sx += min_image(hj.x - h0.x, k.Lx, k.hLx);
    sy += min_image(hj.y - h0.y, k.Ly, k.hLy);
  }
  const double cx = wrap_box(h0.x + sx / (double)n, k.Lx), cy = wrap_box(h0.y + sy / (double)n, k.Ly);
  const int t = d.ctag[c];
  key[t] = key_of_position(cx, cy, k, m);
  val[t] = c;
}

// ---- stable LSD radix sort, one 8-bit digit per pass -----------------------------------------
__global__ void __launch_bounds__(32 * kWarpsPerBlock)
radix_hist_kernel(const unsigned int* __restrict__ key, int n, int shift, int n_seg, unsigned int* __restrict__ hist) {
  __shared__ unsigned int cnt[kWarpsPerBlock][256];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int seg = blockIdx.x * kWarpsPerBlock + warp;
  for (int i = lane; i < 256; i += 32) cnt[warp][i] = 0;
  __syncwarp();
  if (seg < n_seg) {
    const int beg = seg * kSeg, end = min(n, beg + kSeg);
    for (int i = beg + lane; i < end; i += 32) atomicAdd(&cnt[warp][(key[i] >> shift) & 255u], 1u);
  }
  __syncwarp();
  if (seg < n_seg)
    for (int i = lane; i < 256; i += 32) hist[(size_t)i * n_seg + seg] = cnt[warp][i];
}

// exclusive scan of `len` counters by one block (len is at most a few million; off the hot path)
__global__ void __launch_bounds__(1024)
exclusive_scan_kernel(unsigned int* __restrict__ a, long long len) {
  __shared__ unsigned int part[1024];
  const long long chunk = (len + 1023) / 1024;
  const long long beg = (long long)threadIdx.x * chunk, end = min(len, beg + chunk);
  unsigned int s = 0;
  for (long long i = beg; i < end; ++i) s += a[i];
  part[threadIdx.x] = s;
  __syncthreads();
  // Hillis-Steele inclusive scan of the 1024 partial sums
  for (int off = 1; off < 1024; off <<= 1) {
    unsigned int v = threadIdx.x >= off ? part[threadIdx.x - off] : 0u;
    __syncthreads();
    part[threadIdx.x] += v;
    __syncthreads();
  }
  unsigned int run = threadIdx.x ? part[threadIdx.x - 1] : 0u;
  for (long long i = beg; i < end; ++i) { const unsigned int t = a[i]; a[i] = run; run += t; }
}

__global__ void __launch_bounds__(32 * kWarpsPerBlock)
radix_scatter_kernel(const unsigned int* __restrict__ key_in, const int* __restrict__ val_in, int n, int shift, int n_seg,
                     const unsigned int* __restrict__ hist, unsigned int* __restrict__ key_out, int* __restrict__ val_out) {
  __shared__ unsigned int base[kWarpsPerBlock][256];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int seg = blockIdx.x * kWarpsPerBlock + warp;
  if (seg >= n_seg) return;
  for (int i = lane; i < 256; i += 32) base[warp][i] = hist[(size_t)i * n_seg + seg];
  __syncwarp();
  const int beg = seg * kSeg, end = min(n, beg + kSeg);
  for (int i0 = beg; i0 < end; i0 += 32) {
    const int i = i0 + lane;
    const bool valid = i < end;
    const unsigned int active = __ballot_sync(0xffffffffu, valid);
    if (valid) {
      const unsigned int kx = key_in[i];
      const int vx = val_in[i];
      const unsigned int dg = (kx >> shift) & 255u;
      const unsigned int peers = __match_any_sync(active, dg);
      const unsigned int rank = __popc(peers & ((1u << lane) - 1u));
      const unsigned int b = base[warp][dg];
      __syncwarp(active);
      if (rank == 0) base[warp][dg] = b + __popc(peers);
      __syncwarp(active);
      key_out[b + rank] = kx;
      val_out[b + rank] = vx;
    }
  }
}

__global__ void invert_kernel(const int* __restrict__ order, int n, int* __restrict__ newidx) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) newidx[order[i]] = i;
}

// ---- apply the permutation ---------------------------------------------------------------------
__global__ void permute_vertices_kernel(const Dev a, const Dev b, const Consts k, const int* __restrict__ order_v,
                                        const int* __restrict__ newidx_v, const int* __restrict__ newidx_c) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= k.V) return;
  const int o = order_v[i];
  b.pos[i] = a.pos[o];
  b.vtag[i] = a.vtag[o];
#pragma unroll
  for (int s = 0; s < 3; ++s) {
    b.vn[s * k.Vs + i] = newidx_v[a.vn[s * k.Vs + o]];
    b.vc[s * k.Vs + i] = newidx_c[a.vc[s * k.Vs + o]];
  }
}

__global__ void permute_cells_kernel(const Dev a, const Dev b, const Consts k, const int* __restrict__ order_c,
                                     const int* __restrict__ newidx_v) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= k.N) return;
  const int o = order_c[i];
  const int n = a.cvn[o];
  b.cvn[i] = n;
  b.theta[i] = a.theta[o];
  b.rec[i] = a.rec[o];
  b.ctag[i] = a.ctag[o];
  for (int q = 0; q < k.S / 4; ++q) {
    const int4 src = a.cv[(size_t)q * k.N + o];
    int4 dst;
    // padding entries repeat entry 0, so every entry is a valid index
    dst.x = newidx_v[src.x]; dst.y = newidx_v[src.y]; dst.z = newidx_v[src.z]; dst.w = newidx_v[src.w];
    b.cv[(size_t)q * k.N + i] = dst;
  }
}

size_t sort_hist_entries(int n) { return (size_t)256 * (size_t)((n + kSeg - 1) / kSeg); }

static inline int cdiv(long long a, int b) { return (int)((a + b - 1) / b); }

// sort (key,val) pairs held in sc.key[0]/sc.val[0]; returns the buffer index holding the result
static int radix_sort_pairs(const SortScratch& sc, int n, int key_bits, cudaStream_t s, int* launches) {
  const int n_seg = (n + kSeg - 1) / kSeg;
  int cur = 0;
  for (int shift = 0; shift < key_bits; shift += 8) {
    radix_hist_kernel<<<cdiv(n_seg, kWarpsPerBlock), 32 * kWarpsPerBlock, 0, s>>>(sc.key[cur], n, shift, n_seg, sc.hist);
    exclusive_scan_kernel<<<1, 1024, 0, s>>>(sc.hist, (long long)256 * n_seg);
    radix_scatter_kernel<<<cdiv(n_seg, kWarpsPerBlock), 32 * kWarpsPerBlock, 0, s>>>(
        sc.key[cur], sc.val[cur], n, shift, n_seg, sc.hist, sc.key[1 - cur], sc.val[1 - cur]);
    cur = 1 - cur;
    *launches += 3;
  }
  return cur;
}

int hilbert_bits(const Consts& k) {
  // grid spacing <= 0.5 in units of the mean cell size (sqrt of box area / N), 1 <= m <= 16
  const double L = k.Lx > k.Ly ? k.Lx : k.Ly;
  const double unit = sqrt(k.Lx * k.Ly / (double)k.N);
  int m = 1;
  while (m < 16 && L / (double)(1u << m) > 0.5 * unit) ++m;
  return m;
}

int launch_hilbert_sort(const Dev& a, const Dev& b, const Consts& k, const SortScratch& sc, cudaStream_t s) {
  int launches = 0;
  const int m = hilbert_bits(k);
  // vertices
  vertex_keys_kernel<<<cdiv(k.V, 256), 256, 0, s>>>(a, k, m, sc.key[0], sc.val[0]);
  ++launches;
  int r = radix_sort_pairs(sc, k.V, 2 * m, s, &launches);
  cudaMemcpyAsync(sc.order_v, sc.val[r], sizeof(int) * (size_t)k.V, cudaMemcpyDeviceToDevice, s);
  invert_kernel<<<cdiv(k.V, 256), 256, 0, s>>>(sc.order_v, k.V, sc.newidx_v);
  ++launches;
  // cells
  cell_keys_kernel<<<cdiv(k.N, 256), 256, 0, s>>>(a, k, m, sc.key[0], sc.val[0]);
  ++launches;
  r = radix_sort_pairs(sc, k.N, 2 * m, s, &launches);
  cudaMemcpyAsync(sc.order_c, sc.val[r], sizeof(int) * (size_t)k.N, cudaMemcpyDeviceToDevice, s);
  invert_kernel<<<cdiv(k.N, 256), 256, 0, s>>>(sc.order_c, k.N, sc.newidx_c);
  ++launches;
  permute_vertices_kernel<<<cdiv(k.V, 256), 256, 0, s>>>(a, b, k, sc.order_v, sc.newidx_v, sc.newidx_c);
  permute_cells_kernel<<<cdiv(k.N, 256), 256, 0, s>>>(a, b, k, sc.order_c, sc.newidx_v);
  launches += 2;
  return launches;
}

unsigned int hilbert_index_host(unsigned int x, unsigned int y, int m) { return hilbert_index(x, y, m); }

// test hook: Hilbert indices of explicit grid coordinates
__global__ void hilbert_index_kernel(int m, long long n, const unsigned int* ix, const unsigned int* iy, unsigned int* out) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = hilbert_index(ix[i], iy[i], m);
}
int launch_hilbert_index(int m, long long n, const unsigned int* ix, const unsigned int* iy, unsigned int* out, cudaStream_t s) {
  if (n <= 0) return 0;
  hilbert_index_kernel<<<cdiv(n, 256), 256, 0, s>>>(m, n, ix, iy, out);
  return 1;
}

}  // namespace avm
