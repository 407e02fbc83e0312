// avm_forces_static.cu — avm_forces_static: geometry + vertex forces of a tiling for callers that cannot
// allocate device memory (see include/avm.h for who they are and for the contract).
//
// The ordinary path (avm_create + avm_compute_forces) keeps the per-cell areas and perimeters between its two
// kernels in the caller's workspace, and building an avm_sim allocates host memory.  Here the same two kernels
// read the caller's user-order arrays directly and hand the per-cell (A, P) pairs over through g_static_ap, a
// fixed-size array that is part of the library's device image: it exists from the moment the module is loaded
// on a GPU until the process exits, on every GPU that loads the library, whether this file is used or not.
//
// Host code must never pass `g_static_ap` itself to a kernel: in host code that name is a host-side handle of
// the symbol, not a device address.  static_ap_on() asks the runtime for the device address
// (cudaGetSymbolAddress), once per device, with that device current, and that address is what the kernels get.
#include <mutex>
#include "avm_internal.cuh"

namespace avm {
void note_cuda_error(const char* call, cudaError_t e);   // avm_api.cu: text behind avm_last_cuda_error()
}

using namespace avm;

// (A_c, P_c) of every cell of the call in progress: 16 bytes x 65536 cells = 1 MiB per GPU.
static __device__ __align__(256) double2 g_static_ap[AVM_FORCES_STATIC_MAX_CELLS];

namespace {

constexpr int kStaticMaxCells = AVM_FORCES_STATIC_MAX_CELLS;
constexpr int kStaticMaxDevices = 64;

std::mutex g_static_mu;                               // guards the table below (constexpr constructor: no allocation)
double2* g_static_ap_dev[kStaticMaxDevices] = {};     // device address of g_static_ap on each device, once known

// Device address of g_static_ap on `device`, which must be the current device.  The first call on a device
// resolves the symbol (this loads the module there if it is not loaded yet), later calls return the cached address.
cudaError_t static_ap_on(int device, double2** out) {
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_ap_dev[device]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_static_ap);
    if (e != cudaSuccess) return e;
    g_static_ap_dev[device] = (double2*)p;
  }
  *out = g_static_ap_dev[device];
  return cudaSuccess;
}

// Vertex j of a user-order position array [V][2]; two scalar loads, the caller's pointer need only be 8-byte aligned.
__device__ __forceinline__ double2 user_pos(const double* __restrict__ pos_xy, int v) {
  return make_double2(pos_xy[2 * (size_t)v], pos_xy[2 * (size_t)v + 1]);
}

// Row a1 (Eq. A1 inputs, R14): area and perimeter of cell c from its user-order row, summed with
// geom_edge in the order cell_area_perimeter uses, so the bits equal those of avm_compute_forces.
__global__ void static_geometry_kernel(const double* __restrict__ pos_xy, const int* __restrict__ cvn,
                                       const int* __restrict__ cv, const Consts k, double2* __restrict__ ap,
                                       double* __restrict__ ap_user) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= k.N) return;
  const int* row = cv + (size_t)c * k.S;
  const int n = cvn[c];
  const double2 h0 = user_pos(pos_xy, row[0]);
  double rxp = 0.0, ryp = 0.0, acc = 0.0, per = 0.0;
  for (int j = 1; j <= n; ++j) {
    double rx = 0.0, ry = 0.0;
    if (j < n) {
      const double2 hj = user_pos(pos_xy, row[j]);
      rx = min_image(__dsub_rn(hj.x, h0.x), k.Lx, k.hLx);
      ry = min_image(__dsub_rn(hj.y, h0.y), k.Ly, k.hLy);
    }
    geom_edge(rxp, ryp, rx, ry, acc, per);
    rxp = rx; ryp = ry;
  }
  const double A = __dmul_rn(0.5, acc);
  ap[c] = make_double2(A, per);
  if (ap_user) { ap_user[2 * (size_t)c] = A; ap_user[2 * (size_t)c + 1] = per; }
}

// Row a2 (Eq. A2-A5): force on vertex v from its three neighbours and the (A, P) of its three
// cells, which the geometry kernel of the same call left in `ap`.  User-order lists [V][3].
__global__ void static_forces_kernel(const double* __restrict__ pos_xy, const int* __restrict__ vn,
                                     const int* __restrict__ vc, const Consts k, const double2* __restrict__ ap,
                                     double* __restrict__ force_xy) {
  const int v = blockIdx.x * blockDim.x + threadIdx.x;
  if (v >= k.V) return;
  const double2 h = user_pos(pos_xy, v);
  CellRec c[3];
  double2 q[3];
#pragma unroll
  for (int s = 0; s < 3; ++s) {
    q[s] = user_pos(pos_xy, vn[3 * (size_t)v + s]);
    const double2 a = ap[vc[3 * (size_t)v + s]];
    c[s].a = k.KA2 * (a.x - k.A0); c[s].p = k.KP2 * (a.y - k.P0);
    c[s].nx = 0.0; c[s].ny = 0.0;
  }
  const double2 f = vertex_force(h, q[0], q[1], q[2], c[0], c[1], c[2], k);
  force_xy[2 * (size_t)v] = f.x; force_xy[2 * (size_t)v + 1] = f.y;
}

}  // namespace

#define AVM_STATIC_CUDA(call)                      \
  do {                                             \
    const cudaError_t e_ = (call);                 \
    if (e_ != cudaSuccess) {                       \
      note_cuda_error(#call, e_);                  \
      return AVM_ECUDA;                            \
    }                                              \
  } while (0)

extern "C" int avm_forces_static(const avm_params* p, const double* pos_xy, const int32_t* cell_vertex_num,
                                 const int32_t* cell_vertices, const int32_t* vertex_neighbors,
                                 const int32_t* vertex_cell_neighbors, double* force_xy, double* area_perim,
                                 void* cuda_stream) {
  if (!p || !pos_xy || !cell_vertex_num || !cell_vertices || !vertex_neighbors || !vertex_cell_neighbors) return AVM_EINVAL;
  if (!force_xy && !area_perim) return AVM_EINVAL;
  if (p->n_cells < 4 || p->n_vertices != 2 * (int64_t)p->n_cells) return AVM_EINVAL;
  if (p->max_cell_vertices < 8 || p->max_cell_vertices > 32 || (p->max_cell_vertices & 3)) return AVM_EINVAL;
  if (!(p->Lx > 0.0) || !(p->Ly > 0.0)) return AVM_EINVAL;
  if (p->device < 0 || p->device >= kStaticMaxDevices) return AVM_EINVAL;
  if (p->n_cells > kStaticMaxCells) return AVM_ETOOLARGE;   // the static array holds no more; use avm_compute_forces
  AVM_STATIC_CUDA(cudaSetDevice(p->device));
  double2* ap = nullptr;
  AVM_STATIC_CUDA(static_ap_on(p->device, &ap));
  Consts k = {};
  k.N = p->n_cells; k.V = p->n_vertices; k.S = p->max_cell_vertices;
  k.Lx = p->Lx; k.Ly = p->Ly; k.hLx = 0.5 * p->Lx; k.hLy = 0.5 * p->Ly;
  k.KA = p->KA; k.KP = p->KP; k.KA2 = 2.0 * p->KA; k.KP2 = 2.0 * p->KP; k.A0 = p->A0; k.P0 = p->P0;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  // Nothing in g_static_ap has to start at zero: the geometry kernel overwrites entries 0..N-1 and the force
  // kernel, ordered behind it on the stream, reads only those.  Whatever an earlier call left beyond N is never read.
  static_geometry_kernel<<<(k.N + 127) / 128, 128, 0, s>>>(pos_xy, cell_vertex_num, cell_vertices, k, ap, area_perim);
  if (force_xy)
    static_forces_kernel<<<(k.V + 255) / 256, 256, 0, s>>>(pos_xy, vertex_neighbors, vertex_cell_neighbors, k, ap, force_xy);
  AVM_STATIC_CUDA(cudaPeekAtLastError());
  return AVM_OK;
}
