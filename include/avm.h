/* avm.h — C ABI of the B200-native active-vertex-model (AVM) hot path.
 *
 * One overdamped timestep of a 3-coordinated polygonal tiling in a periodic box, as defined by
 * arXiv:1702.02939 ("cellGPU", D. M. Sussman); citations below are lines of
 * /root/reference/PAPER.md with the section/equation they fall in.  R-numbers refer to the
 * readings of the paper listed in DESIGN.md.
 *
 *   state    : vertex positions h_v in [0,Lx)x[0,Ly); cell directors theta_c; the three flat
 *              topology lists of PAPER.md:66 (§II.B): vertices around each cell in
 *              counter-clockwise order, vertices each vertex is connected to, cells that border
 *              each vertex.
 *   one step : geometry of every cell -> force on every vertex -> move the vertices (Eq. 4) ->
 *              rotate the directors -> one T1 pass on the moved positions
 *              (PAPER.md:62-64 §II.B, :104-108 §II.D).
 *
 * Conventions common to every entry point
 *   - Plain C, no exceptions cross the boundary.  Return 0 on success, a negative AVM_E* code
 *     otherwise; avm_strerror() names it.
 *   - "device pointer" = CUDA global memory on params.device; "host pointer" = ordinary (pageable
 *     or pinned) host memory.  The *_host twins take host pointers and do the copies themselves.
 *   - The library never allocates or frees device memory: the caller passes one workspace of
 *     avm_workspace_bytes() bytes (256-byte aligned) that must outlive the avm_sim.  The avm_sim
 *     object itself owns only host-side bookkeeping: a heap object and, when the kernel schedule is
 *     chosen per step (the default from a million vertices), one 64-byte block of mapped pinned host
 *     memory (cudaHostAlloc) through which the kernels report the T1 load; avm_destroy frees both.
 *     avm_forces_static (below) allocates nothing at all.
 *   - All work is enqueued on the CUDA stream given at creation.  avm_step never synchronises the
 *     host (the AVM loop has no host<->device traffic).
 *   - Every user-visible array is in USER ORDER (the order given to avm_create), whatever the
 *     internal Hilbert order is.  Index layout, all C-contiguous:
 *       pos_xy                [V][2] double   vertex positions
 *       cell_vertex_num       [N]    int32    number of vertices of each cell (3..S)
 *       cell_vertices         [N][S] int32    CCW vertex list of each cell, unused slots = -1
 *       vertex_neighbors      [V][3] int32    the three vertices joined to v, CCW around v
 *       vertex_cell_neighbors [V][3] int32    slot k = the cell between edges (v,n_k), (v,n_k+1),
 *                                             i.e. in that cell's row (n_k+1, v, n_k) are consecutive
 *       theta                 [N]    double   director angle of each cell (not wrapped)
 *     Any OUTPUT pointer may be NULL (that array is skipped).
 */
#ifndef AVM_H_
#define AVM_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct avm_sim avm_sim; /* opaque */

typedef struct avm_params {
  int32_t n_cells;           /* N                                                               */
  int32_t n_vertices;        /* V, must equal 2N (3-coordinated tiling of the torus)            */
  int32_t max_cell_vertices; /* S: row stride of cell_vertices, 8..32, multiple of 4            */
  int32_t sort_every;        /* 0 = never; k > 0 = Hilbert re-sort after every k-th step        */
  double Lx, Ly;             /* periodic box (R13); every cell must stay narrower than L/2      */
  double KA, KP, A0, P0;     /* Eq. A1: E = sum KA (A-A0)^2 + KP (P-P0)^2        */
  double v0, Dr, mu, dt;     /* Eq. 4, director noise variance 2 Dr */
  double l_c;                /* T1 threshold: edges with length < l_c are flipped (R9)          */
  uint64_t seed;             /* Philox4x32-10 key (R16)                                         */
  uint64_t step0;            /* step counter at creation; resume from a saved state is exact    */
  int32_t device;            /* CUDA device ordinal                                             */
  int32_t flags;             /* AVM_FLAG_*                                                      */
} avm_params;

enum {
  AVM_FLAG_SORT_AT_CREATE = 1, /* Hilbert-order cells and vertices once inside avm_create       */
  /* Kernel schedule.  Default: chosen from the system size and, per step, from the T1 load.
   * FUSED: two launches per step, the T1 flips of a step run inside the next force/move launch.
   * UNFUSED: three launches per step, a stand-alone T1 kernel.  PERSISTENT: one cooperative launch
   * per avm_step call (per stretch between re-sorts) advances all its steps, with grid-wide barriers
   * between the stages (launch-free stepping; the default for systems of at most 8192 vertices: one
   * CTA up to 512 vertices, one thread-block cluster with the hardware cluster barrier beyond).  All
   * schedules give the same bits (tests); at most one flag may be given. */
  AVM_FLAG_SCHEDULE_FUSED = 4,
  AVM_FLAG_SCHEDULE_UNFUSED = 8,
  AVM_FLAG_SCHEDULE_PERSISTENT = 16,
  /* bits 8..15: maximum number of T1 passes per step.  0 or 1 = one pass per step (the rule of
   * BASELINE.json's north_star, the default and the timed path).  P > 1 = the paper's own rule
   * (the T1 kernel is "called repeatedly until no changes"): after the first pass
   * the detect / resolve / flip passes are repeated on the current state until a pass finds no
   * candidate, at most P passes in total. */
  AVM_FLAG_T1_PASSES_SHIFT = 8,
  AVM_FLAG_T1_PASSES_MASK = 0xff00
};

/* Counters since creation.  error is a sticky bit set: 1 = a non-finite position was produced,
 * 2 = a flip was suppressed because a cell row would exceed S, 4 = the lists given to avm_create
 * are out of range or inconsistent (avm_create then fails with AVM_EINCONSISTENT), 8 = a T1
 * candidate list overflowed its capacity (cannot happen for a valid tiling), 16 = the driver refused
 * the launch-free persistent kernel (e.g. the GPU is shared and the grid cannot be co-resident) and the
 * run went on with one launch per kernel: same results, more launches. */
typedef struct avm_stats {
  int64_t step;             /* current step counter (step0 + steps taken)                       */
  int64_t t1_short;         /* edges found shorter than l_c                                      */
  int64_t t1_candidates;    /* of those, eligible (R10)                                          */
  int64_t t1_flips;         /* candidates that won the conflict rule (R11) and were flipped      */
  int64_t t1_blocked;       /* candidates blocked by a smaller key sharing a cell                */
  int64_t overflow_rejects; /* short edges rejected because an end cell is already at S          */
  int64_t error;            /* sticky error bits                                                 */
  int64_t n_sorts;          /* Hilbert re-sorts done                                             */
  int64_t kernel_launches;  /* kernels this library has launched since creation                  */
} avm_stats;

enum {
  AVM_OK = 0,
  AVM_EINVAL = -1,        /* NULL / out-of-range argument, V != 2N, bad stride                   */
  AVM_EWORKSPACE = -2,    /* workspace too small or misaligned                                   */
  AVM_EINCONSISTENT = -3, /* the topology lists contradict each other or a row is out of range   */
  AVM_ECUDA = -4,         /* a CUDA call failed; avm_last_cuda_error() has the text              */
  AVM_ENOMEM = -5,
  AVM_ETOOLARGE = -6      /* avm_forces_static: more cells than AVM_FORCES_STATIC_MAX_CELLS             */
};

/* Bytes of device workspace avm_create needs for these parameters (0 on invalid parameters). */
size_t avm_workspace_bytes(const avm_params* params);

/* Build a simulation from an initial state (PAPER.md:66 lists; theta: PAPER.md:50).
 * Inputs are copied into the workspace; the caller keeps ownership of its arrays.  The lists are
 * validated on the device (ranges, slot convention of vertex_cell_neighbors against the rows);
 * avm_create synchronises the stream once to report AVM_EINCONSISTENT.
 * avm_create: all array arguments are device pointers.  avm_create_host: host pointers. */
int avm_create(const avm_params* params, const double* pos_xy, const int32_t* cell_vertex_num,
               const int32_t* cell_vertices, const int32_t* vertex_neighbors,
               const int32_t* vertex_cell_neighbors, const double* theta, void* workspace,
               size_t workspace_bytes, void* cuda_stream, avm_sim** out);
int avm_create_host(const avm_params* params, const double* pos_xy, const int32_t* cell_vertex_num,
                    const int32_t* cell_vertices, const int32_t* vertex_neighbors,
                    const int32_t* vertex_cell_neighbors, const double* theta, void* workspace,
                    size_t workspace_bytes, void* cuda_stream, avm_sim** out);

/* Advance n_steps timesteps (order R6).  Asynchronous: only enqueues
 * kernels (and, every sort_every steps, the Hilbert re-sort) on the stream.
 * Conditions arising inside a step set avm_stats.error; they do not stop the run. */
int avm_step(avm_sim* sim, int64_t n_steps);

/* Same steps as avm_step, one launch per kernel (with avm_step's choice between two and three launches
 * per step; never the launch-free persistent kernel, which has no kernel boundaries: for systems that
 * avm_step advances launch-free the times describe the launched schedule instead).  Every kernel of the
 * step is bracketed by CUDA events on the stream and the call synchronises after each step: ms_per_kernel (HOST pointer,
 * [AVM_K_COUNT]) receives the summed device time of each kernel class over the n_steps.  In the
 * default two-launch schedule the T1 flips of a step run inside the next force/move launch, so
 * AVM_K_T1_FLIP only holds the stand-alone T1 kernel that completes the last step.  Measurement
 * aid for the roofline figures of bench.py; not the timed path. */
enum { AVM_K_FORCE_MOVE = 0, AVM_K_CELL_UPDATE = 1, AVM_K_T1_FLIP = 2, AVM_K_COUNT = 3 };
int avm_step_profile(avm_sim* sim, int64_t n_steps, double* ms_per_kernel);

/* Geometry + forces of the current state, nothing modified (App. A.1, Eq. A1-A5):
 * force_xy [V][2] = -dE/dh_v, area_perim [N][2] = (A_c, P_c), user order.  Asynchronous for the
 * device variant; the host variant returns after the copies have completed. */
int avm_compute_forces(avm_sim* sim, double* force_xy, double* area_perim);
int avm_compute_forces_host(avm_sim* sim, double* force_xy, double* area_perim);

/* Geometry and forces of a tiling WITHOUT an avm_sim, a workspace or any allocation — for callers that
 * are not allowed to allocate: code running inside someone else's memory plan (a plugin or a callback of
 * a host application that hands out fixed device buffers and forbids cudaMalloc, which would also
 * synchronise the whole device under the host's feet), real-time loops that must not take the
 * allocator's locks, and processes whose device memory is fully reserved by another pool.  Such a caller
 * cannot provide avm_create's workspace either if nobody gave it one.  Same result as avm_create +
 * avm_compute_forces with the uniform A0, P0, KA, KP of `params` (App. A.1, Eq. A1-A5), to
 * the last bit in the f64 library.
 *
 *   params   : n_cells, n_vertices, max_cell_vertices, Lx, Ly, KA, KP, A0, P0 and device are read; the rest is
 *              ignored.  The call makes params->device the current device, as avm_create does.
 *   inputs   : DEVICE pointers, the user-order arrays of the table above (pos_xy, cell_vertex_num,
 *              cell_vertices, vertex_neighbors, vertex_cell_neighbors), read only, not validated.
 *   outputs  : DEVICE pointers owned by the caller: force_xy [V][2] = -dE/dh_v, area_perim [N][2] = (A_c, P_c);
 *              either may be NULL, not both.
 *   stream   : the two kernels are enqueued on cuda_stream; the call does not synchronise.
 *
 * The per-cell (A, P) pairs travel from the geometry kernel to the force kernel through a fixed array
 * built into the library's device image: 16 bytes x AVM_FORCES_STATIC_MAX_CELLS = 1 MiB of device
 * memory on every GPU that loads the library, held until the process exits.  Consequences:
 *   - n_cells > AVM_FORCES_STATIC_MAX_CELLS is refused with AVM_ETOOLARGE (nothing is enqueued); larger
 *     tilings need avm_compute_forces and a workspace.
 *   - The first call on each device looks the array's device address up (one cudaGetSymbolAddress, which
 *     loads the library's kernels on that device if nothing has yet); make that first call before any
 *     stream capture begins.  Later calls only enqueue the two kernels.
 *   - No call here uses cudaMalloc, cudaFree, cudaHostAlloc or a library routine that allocates.
 *   - All calls on a device share the one array, and it keeps what the last call wrote.  Nothing in it
 *     needs clearing: every entry the force kernel reads was written by the geometry kernel of the same
 *     call.  But two calls whose kernels can run at the same time on one GPU (different streams, or
 *     different host threads on different streams) overwrite each other's (A, P) and give wrong forces:
 *     keep calls on one stream, or order them yourself.
 * Errors: AVM_EINVAL (NULL input, both outputs NULL, V != 2N, bad stride or box, device outside 0..63),
 * AVM_ETOOLARGE, AVM_ECUDA. */
#define AVM_FORCES_STATIC_MAX_CELLS 65536
int avm_forces_static(const avm_params* params, const double* pos_xy, const int32_t* cell_vertex_num,
                      const int32_t* cell_vertices, const int32_t* vertex_neighbors,
                      const int32_t* vertex_cell_neighbors, double* force_xy, double* area_perim,
                      void* cuda_stream);

/* Total energy of the current state, Eq. 1 / A1, summed on the device in a
 * fixed order (deterministic).  energy is a HOST pointer; synchronises the stream. */
int avm_energy(avm_sim* sim, double* energy);

/* Per-cell preferred area and perimeter A_{0,i}, P_{0,i} of Eq. 1 (SURVEY.md
 * section 8(f), NEXT-4) instead of the uniform A0, P0 of Eq. A1.  area0, perimeter0: DEVICE
 * pointers, [N] each, user order, copied; both NULL restores the uniform values of avm_params.
 * Asynchronous.  The values are not part of avm_get_state: a resumed run sets them again. */
int avm_set_cell_targets(avm_sim* sim, const double* area0, const double* perimeter0);

/* Per-cell moduli K_{A,i}, K_{P,i}: Eq. 1 read with the moduli inside the sum,
 * E = sum_i K_{A,i} (A_i - A_{0,i})^2 + K_{P,i} (P_i - P_{0,i})^2.
 * KA, KP: DEVICE pointers, [N] each, user order, copied; both NULL restores the uniform moduli of
 * avm_params.  Independent of avm_set_cell_targets.  Asynchronous; not part of avm_get_state. */
int avm_set_cell_moduli(avm_sim* sim, const double* KA, const double* KP);

/* Observables of the current state, reduced on the device in a
 * fixed order (deterministic): the energy of Eq. 1, the area and perimeter totals, the mean shape
 * index <P / sqrt(A)> over the cells with A > 0 (the order parameter of the rigidity transition
 * the paper's model is used for), area extremes and variance, the number of cells
 * with non-positive signed area (transiently possible, R14), and the running T1 count.
 * out is a HOST pointer; synchronises the stream. */
typedef struct avm_observables {
  double energy, sum_area, sum_perimeter, mean_shape_index, area_min, area_max, area_variance;
  int64_t n_nonpositive_area, step, t1_flips;
  double msd; /* mean-square displacement of the vertices since the reference time (below) */
} avm_observables;
int avm_observe(avm_sim* sim, avm_observables* out);

/* Advance n_steps >= 1 timesteps like avm_step and observe WITHOUT an extra pass over the state
 * ("reductions fused into the geometry pass"): the geometry pass of the
 * last step, which computes every cell's area and perimeter anyway, also reduces the
 * observables, in a fixed order (deterministic).  They therefore describe the MOVED tiling of that
 * step - after its vertex move and director update, before its T1 pass (PAPER.md:62-64 order) -
 * whereas avm_observe describes the state between steps; the two agree whenever the step flips
 * nothing.  out->step and out->t1_flips are read after the step.  out is a HOST pointer;
 * synchronises the stream. */
int avm_step_observe(avm_sim* sim, int64_t n_steps, avm_observables* out);

/* Mean-square displacement (the fluid/solid diagnostic of the regimes of
 * PAPER.md:114-116): <|U_v(t) - U_v(t_ref)|^2> over all vertices, U = unwrapped position.  The library
 * counts, per vertex, the box lengths it has left through the boundary (in the move of Eq. 4 and
 * in the repositioning of a T1), so U = position + count x L costs nothing per step.  The
 * reference time is avm_create / avm_set_positions, or the latest avm_msd_reset.  Neither the counts
 * nor the reference are part of avm_get_state: a resumed run measures from its own creation. */
int avm_msd_reset(avm_sim* sim);

/* Copy the current state out in user order.  stats (HOST pointer, may be NULL) receives the
 * counters; when it is non-NULL, or for the host variant, the call synchronises the stream. */
int avm_get_state(avm_sim* sim, double* pos_xy, int32_t* cell_vertex_num, int32_t* cell_vertices,
                  int32_t* vertex_neighbors, int32_t* vertex_cell_neighbors, double* theta,
                  avm_stats* stats);
int avm_get_state_host(avm_sim* sim, double* pos_xy, int32_t* cell_vertex_num, int32_t* cell_vertices,
                       int32_t* vertex_neighbors, int32_t* vertex_cell_neighbors, double* theta,
                       avm_stats* stats);

/* The GPU-only parts of one self-propelled-Voronoi (SPV) step on a FIXED triangulation (SURVEY.md section
 * 8(f) NEXT-4; section II.C, App. A.2 :171-200).  The triangulation is the dual reading of the
 * lists the simulation holds: vertex v <-> Delaunay triangle with corners
 * vertex_cell_neighbors[v], row c of cell_vertices = the Voronoi vertices around cell c.  cell_xy: DEVICE
 * pointer, [N][2] doubles in USER order, in [0,Lx)x[0,Ly), owned by the caller; a Voronoi start is the tiling
 * whose vertices are the circumcentres of cell_xy.  The repair of an invalid triangulation (CPU/CGAL in the
 * paper, :96-100) is out of scope: these calls never change the lists.  All pointers DEVICE unless stated.
 *
 * avm_spv_geometry: Voronoi vertex of every triangle = circumcentre of its three cells,
 *   stored as the simulation's vertex positions (as avm_set_positions would: the mean-square displacement
 *   of avm_observe restarts from them, which also holds after avm_spv_forces / avm_spv_step) and, if non-NULL, in
 *   voronoi_xy [V][2]; area_perim [N][2] (may be NULL) = (A_c, P_c) of the resulting cells.  Asynchronous.
 * avm_spv_forces (Eq. A6-A7): force_xy [N][2] = -dE/dr_i with E of Eq. 1; force_sets
 *   [N][S][2] (may be NULL) = the contribution of each Voronoi vertex of the row of cell i ("force
 *   sets"; unused slots 0); the force is their sum in row order.  Asynchronous.
 * avm_spv_step (Eq. 3): n_steps times geometry -> forces -> r_i += dt (mu F_i + v0 n_i)
 *   with the director of the start of the step, wrap -> director noise (as in avm_step; the step counter
 *   advances) -> empty-circumcircle test.  n_failed: HOST pointer to two int64: [0] = circumcircle tests
 *   that failed after the last step, [1] = index (0-based, within this call) of the first step after
 *   which any test failed, -1 if none.  cell_flags [N] int32 (may be NULL): 1 for the corners of every
 *   failing triangle and the intruding cell after the last step ("cells that need an update").
 *   Afterwards the simulation's vertex positions are the Voronoi vertices of the final cells.
 *   Synchronises the stream.
 * avm_spv_test_triangulation: the test alone on cell_xy; n_failed: HOST pointer to one int64.
 *   A triangle's circumcircle is tested, strictly, against the cell opposite each of its three edges
 *   (local Delaunay criterion: no test fails <=> the triangulation is the Delaunay triangulation). */
int avm_spv_geometry(avm_sim* sim, const double* cell_xy, double* voronoi_xy, double* area_perim);
int avm_spv_forces(avm_sim* sim, const double* cell_xy, double* force_xy, double* force_sets);
int avm_spv_step(avm_sim* sim, double* cell_xy, int64_t n_steps, int64_t* n_failed, int32_t* cell_flags);
int avm_spv_test_triangulation(avm_sim* sim, const double* cell_xy, int64_t* n_failed, int32_t* cell_flags);

/* Test hooks, not on the timed path.
 * avm_debug_t1: T1 detection + conflict resolution (R9-R11) on the current state WITHOUT
 *   flipping.  Writes up to `capacity` (tag_min, tag_max) pairs of candidates and of winners to
 *   the HOST arrays cand_pairs / winner_pairs ([capacity][2] int32, unsorted) and the full counts
 *   to *n_cand / *n_win.  Synchronises.
 * avm_t1_pass: one T1 pass (detect, resolve, flip) on the current state, no move.
 * avm_set_positions: overwrite the vertex positions (device pointer, user order) and refresh
 *   the cached cell geometry.
 * avm_resort: force a Hilbert re-sort now. */
int avm_debug_t1(avm_sim* sim, int32_t* cand_pairs, int64_t* n_cand, int32_t* winner_pairs,
                 int64_t* n_win, int64_t capacity);
int avm_t1_pass(avm_sim* sim);
int avm_set_positions(avm_sim* sim, const double* pos_xy);
int avm_resort(avm_sim* sim);

/* Raw Philox4x32-10 words (R16) for (seed, step, cell0 .. cell0+n-1), computed by the same device
 * function the director update uses: out_words is a DEVICE pointer to [n][4] uint32.  Test hook
 * for the bit-exact comparison with the oracle and with cuRAND. */
int avm_philox_words(avm_sim* sim, uint64_t seed, uint64_t step, uint64_t cell0, int64_t n,
                     uint32_t* out_words);

/* Hilbert index (R18) of grid cells (ix[i], iy[i]) on a 2^m x 2^m grid, 1 <= m <= 16, computed by
 * the device function the re-sort uses (ix, iy, out: DEVICE pointers to [n] uint32), and the same
 * function compiled for the host (scalar; needs no GPU).  Test hooks. */
int avm_hilbert_index(avm_sim* sim, int32_t m, int64_t n, const uint32_t* ix, const uint32_t* iy, uint32_t* out);
uint32_t avm_hilbert_index_host(int32_t m, uint32_t ix, uint32_t iy);

void avm_destroy(avm_sim* sim);
const char* avm_strerror(int code);
const char* avm_last_cuda_error(void);

/* Storage precision of the library that was loaded: "f64" (libavm_b200.so, the default and the
 * timed path: positions double2, cell records 4 doubles, everything fp64) or "mixed"
 * (libavm_b200_mixed.so: the same sources and the same C ABI built with -DAVM_MIXED=1; SURVEY.md
 * section 8(f) NEXT-3, after the single-precision variant of PAPER.md:120).
 *
 * The mixed library changes STORAGE only; every arithmetic operation of the step stays fp64:
 *   - positions are held on a fixed-point grid of 2^-32 box lengths per axis (8 bytes per vertex
 *     instead of 16): a position handed to the library, moved by a step or set by a T1 is rounded
 *     to the nearest grid point, an absolute error of at most L * 2^-33 per coordinate
 *     (1.2e-7 at L = 1024, 9.3e-10 at L = 8);
 *   - the cached cell records 2 K_A (A - A0), 2 K_P (P - P0), cos theta, sin theta are floats
 *     (16 bytes per cell instead of 32): a relative error of at most 2^-24 each.
 *   theta, the topology lists, tags, Philox and all user-visible arrays are unchanged (doubles in and out).
 * Accuracy contract against the float64 oracle, from an identical state whose positions lie on
 * the grid (tests/test_gpu_mixed.py):
 *   - areas and perimeters (avm_compute_forces): 1e-10 relative, as in the default library;
 *   - forces of avm_compute_forces: 1e-10 relative (they do not go through the cached records);
 *     the force applied inside avm_step: 1e-6 relative to max(|F_v|, rms |F|);
 *   - one step: positions within L * 2^-32 + 1e-6 dt max|F| of the oracle's for every vertex that no T1
 *     repositioned (the end points of a T1 land on the old edge turned by 90 degrees, and the direction
 *     of an old edge of length l is only defined to (grid unit / l): they stay within the new edge length),
 *     theta within the 1e-8 of the default library;
 *   - T1 candidate and winner sets of the moved state: equal outside the band | l - l_c | < 4 L 2^-32;
 *   - trajectories are not comparable step for step beyond a few T1 events (the model is chaotic);
 *     total area = Lx Ly to 1e-9 relative and all topological invariants hold at any length.
 * The run is deterministic and resumes bit-identically from avm_get_state (exported positions are
 * grid points and pack to themselves). */
const char* avm_precision(void);

#ifdef __cplusplus
}
#endif
#endif /* AVM_H_ */
