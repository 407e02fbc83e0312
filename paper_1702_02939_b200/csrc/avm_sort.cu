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
  const double2 h = pos_ld(d.pos + v, k);
  const int t = d.vtag[v];
  key[t] = key_of_position(h.x, h.y, k, m);
  val[t] = v;
}

__global__ void cell_keys_kernel(const Dev d, const Consts k, int m, unsigned int* __restrict__ key, int* __restrict__ val) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= k.N) return;
  const int n = d.cvn[c];
  const double2 h0 = pos_ld(d.pos + row_entry(d.cv, k.N, c, 0), k);
  double sx = 0.0, sy = 0.0;
  for (int j = 1; j < n; ++j) {
    const double2 hj = pos_ld(d.pos + row_entry(d.cv, k.N, c, j), k);
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

// ---- exclusive scan of the digit counters (digit-major, `len` = 256 * segments), three coalesced
// kernels: per-chunk sums, scan of the chunk sums by one block, per-chunk scan with its offset ----
static constexpr int kScanBlock = 1024;
static constexpr int kScanChunk = 4 * kScanBlock;   // four consecutive counters per thread

__device__ __forceinline__ unsigned int block_exclusive_scan(unsigned int x, unsigned int* warp_sums, unsigned int& total) {
  // exclusive scan of one value per thread over a block of kScanBlock threads
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  unsigned int incl = x;
#pragma unroll
  for (int off = 1; off < 32; off <<= 1) {
    const unsigned int y = __shfl_up_sync(0xffffffffu, incl, off);
    if (lane >= off) incl += y;
  }
  if (lane == 31) warp_sums[warp] = incl;
  __syncthreads();
  if (warp == 0) {
    unsigned int w = warp_sums[lane], wi = w;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
      const unsigned int y = __shfl_up_sync(0xffffffffu, wi, off);
      if (lane >= off) wi += y;
    }
    warp_sums[lane] = wi - w;          // exclusive prefix of the warp sums
    if (lane == 31) warp_sums[32] = wi;
  }
  __syncthreads();
  total = warp_sums[32];
  return warp_sums[warp] + incl - x;
}

__global__ void __launch_bounds__(kScanBlock)
scan_chunk_sums_kernel(const unsigned int* __restrict__ a, long long len, unsigned int* __restrict__ sums) {
  __shared__ unsigned int ws[33];
  const long long i = (long long)blockIdx.x * kScanChunk + 4 * threadIdx.x;
  unsigned int s = 0;
  if (i + 3 < len) { const uint4 v = *reinterpret_cast<const uint4*>(a + i); s = v.x + v.y + v.z + v.w; }
  else for (int j = 0; j < 4; ++j) if (i + j < len) s += a[i + j];
  unsigned int total;
  block_exclusive_scan(s, ws, total);
  if (threadIdx.x == 0) sums[blockIdx.x] = total;
}

__global__ void __launch_bounds__(kScanBlock)
scan_top_kernel(unsigned int* __restrict__ sums, int n) {
  __shared__ unsigned int ws[33];
  unsigned int run = 0;
  for (int base = 0; base < n; base += kScanBlock) {
    const int i = base + threadIdx.x;
    const unsigned int x = i < n ? sums[i] : 0u;
    unsigned int total;
    const unsigned int ex = block_exclusive_scan(x, ws, total);
    if (i < n) sums[i] = run + ex;
    run += total;
    __syncthreads();
  }
}

__global__ void __launch_bounds__(kScanBlock)
scan_apply_kernel(unsigned int* __restrict__ a, long long len, const unsigned int* __restrict__ sums) {
  __shared__ unsigned int ws[33];
  const long long i = (long long)blockIdx.x * kScanChunk + 4 * threadIdx.x;
  uint4 v = make_uint4(0, 0, 0, 0);
  const bool full = i + 3 < len;
  if (full) v = *reinterpret_cast<const uint4*>(a + i);
  else { if (i < len) v.x = a[i]; if (i + 1 < len) v.y = a[i + 1]; if (i + 2 < len) v.z = a[i + 2]; }
  unsigned int total;
  const unsigned int ex = sums[blockIdx.x] + block_exclusive_scan(v.x + v.y + v.z + v.w, ws, total);
  const uint4 o = make_uint4(ex, ex + v.x, ex + v.x + v.y, ex + v.x + v.y + v.z);
  if (full) *reinterpret_cast<uint4*>(a + i) = o;
  else { if (i < len) a[i] = o.x; if (i + 1 < len) a[i + 1] = o.y; if (i + 2 < len) a[i + 2] = o.z; }
}

static int launch_exclusive_scan(unsigned int* a, long long len, cudaStream_t s) {
  const int nb = (int)((len + kScanChunk - 1) / kScanChunk);
  unsigned int* sums = a + ((len + 3) & ~3ll);      // chunk sums live behind the counters (sort_hist_entries)
  scan_chunk_sums_kernel<<<nb, kScanBlock, 0, s>>>(a, len, sums);
  scan_top_kernel<<<1, kScanBlock, 0, s>>>(sums, nb);
  scan_apply_kernel<<<nb, kScanBlock, 0, s>>>(a, len, sums);
  return 3;
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
  if (k.per_cell) b.par[i] = a.par[o];
  b.ctag[i] = a.ctag[o];
  for (int q = 0; q < k.S / 4; ++q) {
    const int4 src = a.cv[(size_t)q * k.N + o];
    int4 dst;
    // padding entries repeat entry 0, so every entry is a valid index
    dst.x = newidx_v[src.x]; dst.y = newidx_v[src.y]; dst.z = newidx_v[src.z]; dst.w = newidx_v[src.w];
    b.cv[(size_t)q * k.N + i] = dst;
  }
}

size_t sort_hist_entries(int n) {
  const size_t len = (size_t)256 * (size_t)((n + kSeg - 1) / kSeg);
  return ((len + 3) & ~(size_t)3) + (len + kScanChunk - 1) / kScanChunk + 4;   // counters + their chunk sums
}

static inline int cdiv(long long a, int b) { return (int)((a + b - 1) / b); }

// sort (key,val) pairs held in sc.key[0]/sc.val[0]; returns the buffer index holding the result
static int radix_sort_pairs(const SortScratch& sc, int n, int key_bits, cudaStream_t s, int* launches) {
  const int n_seg = (n + kSeg - 1) / kSeg;
  int cur = 0;
  for (int shift = 0; shift < key_bits; shift += 8) {
    radix_hist_kernel<<<cdiv(n_seg, kWarpsPerBlock), 32 * kWarpsPerBlock, 0, s>>>(sc.key[cur], n, shift, n_seg, sc.hist);
    *launches += launch_exclusive_scan(sc.hist, (long long)256 * n_seg, s) - 1;
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
