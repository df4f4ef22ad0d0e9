/*
 * shasta.h -- C ABI of libshasta.so: the dimensionally split (3+1)D relativistic SHASTA
 * flux-corrected-transport time step of arXiv:1206.0919 on one NVIDIA B200 (sm_100a).
 *
 * Citations are "PAPER.md:<line>" (the paper's text) and "DESIGN.md n" (this repo).
 *
 * Conventions (all entry points)
 *  - Return 0 on success, <0 on error: SHASTA_EINVAL bad argument, SHASTA_ECUDA CUDA error,
 *    SHASTA_ENOMEM out of device memory, SHASTA_ESTATE wrong state (e.g. step before
 *    set_state).  Nothing throws or aborts; shasta_last_error(h) gives the message.
 *  - Fields are SoA arrays of nx*ny*nz doubles, x fastest: index ix + nx*(iy + ny*iz)
 *    (the paper's flat index).  Field order of conserved fields: E, Mx, My, Mz, R
 *    (R is the paper's N, eq. (9)); of primitives: e, p, n, vx, vy, vz.
 *  - Pointers named *_dev are DEVICE pointers, pointers named *_host are HOST pointers (pinned
 *    or pageable).  The caller owns every buffer it passes; the library copies and never keeps
 *    a caller pointer.  The handle owns all device memory it allocates.
 *  - `stream` is a cudaStream_t passed as void* (NULL = the default stream).  Unless stated
 *    otherwise a call only enqueues work on `stream` and returns; it is the caller's job to
 *    keep the buffers alive until the stream has run.
 *  - There is no CPU fallback: without a CUDA device shasta_create returns SHASTA_ECUDA.
 */
#ifndef SHASTA_H
#define SHASTA_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct shasta shasta_t;   /* opaque */

#define SHASTA_OK      0
#define SHASTA_EINVAL (-1)
#define SHASTA_ECUDA  (-2)
#define SHASTA_ENOMEM (-3)
#define SHASTA_ESTATE (-4)

/* option keys for shasta_set_option */
#define SHASTA_BOUNDARY   0   /* 0 = outflow (default): ghost = copy of the edge cell; 1 = periodic   */
#define SHASTA_EOS_MASS   1   /* m in p = (eos_gamma-1)(e - m n); default 0 -> p = (Gamma-1) e         */
#define SHASTA_PRECISION  2   /* 64 (default) | 32: storage and transport arithmetic (before set_state) */
#define SHASTA_STEP_INDEX 3   /* step counter s indexing the axis table (resume / tests)                */
#define SHASTA_SEGMENT    4   /* tuning: cells marched per work item along the sweep axis (0 = auto)    */
#define SHASTA_VARIANT    5   /* reserved (round 1 had a second kernel family here); only 0 is accepted */

#define SHASTA_NO_TMA     6   /* test hook: 1 = the sweeps fill/drain their shared-memory tiles with cp.async + stores
                                 even where TMA is usable (16 B row strides); same bits either way; default 0 */
#define SHASTA_PREDICTOR  7   /* scheme variant: 0 = R1 (default, reading G4): half step = eq. (17)
                                 alone with lambda/2; 1 = R2: half step = the complete kernel with lambda/2, eq. (17)
                                 and eqs. (18)-(22).  R2 runs the per-cell kernels (one thread per
                                 cell, the paper's own decomposition), fp64 only                      */
#define SHASTA_DIFF       8   /* factor on the antidiffusive flux A^ph of eq. (19) (Listing 1 `diff`);
                                 1 = paper default, 0 = the "n/af" mode; 0 <= diff <= 8            */
#define SHASTA_CELL_PATH  9   /* 1 = per-cell kernels for the default scheme too (A/B datapoint "the paper's design on
                                 this GPU", tests); default 0 = fused sweep kernels                                    */

#define SHASTA_NO_DEFER  10   /* test hook / A-B: 1 = a step whose last sweep runs along x writes its primitives at once with
                                 the element-wise pass; default 0 = shasta_step lets the first sweep of the next step write
                                 them (same values, one pass over the conserved fields less)            */

#define SHASTA_PRIMS_RAW 11   /* test hook: 1 = shasta_get_primitives[_host] copies the primitive fields as they are stored,
                                 without recomputing them when they are stale (reads back what emit_primitives = 2 wrote) */

#define SHASTA_BATCH     12   /* B >= 1 independent events of the same grid advanced together by every launch (the paper's
                                 use case is event-by-event statistics).  Every
                                 field argument then holds B consecutive events, B*nx*ny*nz doubles, event b at offset
                                 b*nx*ny*nz; shasta_conserved_totals writes 5*B values.  Events never interact: each has
                                 its own boundary.  Before the first set_state; default 1                               */

#define SHASTA_GRAPH     13   /* launch mode of shasta_step: 0 = every kernel launched on its own; 1 = whole cycles of the axis
                                 table (6 steps = 18 sweeps for the paper's table) are captured once into a CUDA graph and
                                 replayed; 2 (default) = 1 for grids below 2^22 cells, where a sweep lasts ~10 us and the
                                 "orchestration overhead" of PAPER.md:155 shows, else 0.  Same kernels, same results.  */

#define SHASTA_ANTIDIFFUSION 14 /* 0 (default) = phoenical antidiffusion, eq. (19): A = diff/8 (D^ - 1/8 (D_{j+1} - 2 D_j + D_{j-1}));
                                 1 = explicit antidiffusion, A = diff/8 D^ (differences of the transported-diffused field
                                 only): the variant of PAPER.md:123, footnote 1.  Same kernels: the
                                 coefficient of the second difference is a kernel constant (-1/8 or 0)                 */

#define SHASTA_BOUNDARY_Z 15   /* boundary rule of the z sweeps only: -1 (default) = as SHASTA_BOUNDARY; 0 = outflow, 1 = periodic.
                                 For a rank of a z-slab decomposition: its grid carries 4 halo
                                 planes per neighbour, refreshed with shasta_set_planes before each z sweep, and its z
                                 sweeps run with 0 whatever the global rule is                                           */

/*
 * Create a solver for an nx*ny*nz grid.  The scheme depends on lambda = dt/dx only
 * (eqs. (15)-(17)); dx enters shasta_conserved_totals.  0 < lambda <= 0.5
 * (SHASTA's stability range, the denominators of eq. (15) stay > 0), 1 < eos_gamma < 2 (causal sound speed)
 * (4/3 gives p = e/3).  Allocates 2x5 conserved fields (ping-pong, the paper's double
 * buffering PAPER.md:161) + 6 primitive fields on the current device.
 */
int shasta_create(shasta_t** out, int nx, int ny, int nz, double dx, double lambda, double eos_gamma);
void shasta_destroy(shasta_t* h);

/* Options.  PRECISION, BATCH and EOS_MASS must be set before the first shasta_set_state (SHASTA_ESTATE afterwards);
 * every other option may be changed between calls (it takes effect with the next launch).  A handle belongs to the
 * device that was current at shasta_create: calls made with another device current return SHASTA_ESTATE. */
int shasta_set_option(shasta_t* h, int key, double value);

/* Tabled equation of state (the velocity is found by root finding "to allow
 * for an easy implementation of a tabled equation of state").  p_host: HOST pointer to ne*nn pressures, e fastest:
 * p[i + ne*j] = P(e_i, n_j) at the nodes e_i = i e_max/(ne-1), n_j = j n_max/(nn-1).  Between nodes P is bilinear, outside
 * the table the nearest cell's bilinear form continues (linear extrapolation), and P is floored at 0 (DESIGN.md 3,
 * reading T1 -- the paper prints no table and no interpolation rule).  The table is copied to the device; it replaces
 * eos_gamma / SHASTA_EOS_MASS in every cons2prim of the path and in shasta_set_state.  p_host == NULL: back to the analytic
 * EOS.  Call before shasta_set_state.  The EOS must be causal (0 <= dP/de <= 1) for the velocity root to be unique. */
int shasta_set_eos_table(shasta_t* h, const double* p_host, int ne, int nn, double e_max, double n_max);

/* Axis order: step s runs sweeps along axes[(3s+k) % n], k = 0,1,2 (0=x,1=y,2=z).  Default: the
 * paper's 18-entry table branch[], i.e. the six permutations.  n % 3 == 0, n <= 63.
 * `axes` is a host pointer. */
int shasta_set_sweep_table(shasta_t* h, const int* axes_host, int n);

/* Primitive initial state -> conserved fields, eqs. (9)-(11) PAPER.md:58-62:
 * p = EOS(e,n), w = (e+p)/(1-v^2), E = w - p, M = w v, R = n/sqrt(1-v^2).  Requires |v| < 1.
 * Also fills the primitive output fields (they equal the input up to round-off). */
int shasta_set_state(shasta_t* h, const double* e_dev, const double* n_dev, const double* vx_dev,
                     const double* vy_dev, const double* vz_dev, void* stream);
/* Same with HOST pointers: the host->device copies are enqueued on `stream` (asynchronous only if
 * the host memory is pinned). */
int shasta_set_state_host(shasta_t* h, const double* e_host, const double* n_host,
                          const double* vx_host, const double* vy_host, const double* vz_host,
                          void* stream);
/* Set / get the conserved fields directly (checkpoint-resume, parity on conserved fields).
 * set: all five required; the causality projection Pi (G6-G8) is NOT applied.
 * get: any pointer may be NULL = skip. */
int shasta_set_conserved(shasta_t* h, const double* E_dev, const double* Mx_dev, const double* My_dev,
                         const double* Mz_dev, const double* R_dev, void* stream);
int shasta_get_conserved(shasta_t* h, double* E_dev, double* Mx_dev, double* My_dev, double* Mz_dev,
                         double* R_dev, void* stream);

/*
 * Planes z0 .. z0+nplanes-1 (z is the slowest axis: one contiguous block of nplanes*nx*ny values per field) of the CURRENT
 * conserved state, copied to / from DEVICE arrays of nplanes*nx*ny doubles in field order E, Mx, My, Mz, R (NULL = skip
 * the field).  Asynchronous on `stream`; fp32 storage converts.  For the halo exchange of a z-slab decomposition
 * (SURVEY.md 8(e)): a rank sends the 4 planes next to each interface and writes what it receives into its halo planes
 * before every z sweep (paper_1206_0919_b200/zslab.py).  set_planes invalidates the primitive fields.  SHASTA_ESTATE
 * before the first set_state or with SHASTA_BATCH > 1, SHASTA_EINVAL for planes outside [0, nz).
 */
int shasta_get_planes(shasta_t* h, int z0, int nplanes, double* E_dev, double* Mx_dev, double* My_dev, double* Mz_dev,
                      double* R_dev, void* stream);
int shasta_set_planes(shasta_t* h, int z0, int nplanes, const double* E_dev, const double* Mx_dev, const double* My_dev,
                      const double* Mz_dev, const double* R_dev, void* stream);
/* Zero-copy form of the two calls above: the DEVICE address of plane z0 (0 <= z0 <= nz) of conserved field `field`
 * (0..4 = E, Mx, My, Mz, R) inside the handle's CURRENT state buffer, so that a halo exchange can send from and receive
 * into the planes themselves (ncclSend/ncclRecv, peer copies).  Elements are the storage type (double, or float with
 * SHASTA_PRECISION 32), planes z0.. follow contiguously up to plane nz.  The handle keeps ownership.  The address is
 * valid only until the next shasta_sweep / shasta_step / shasta_set_* call on the handle (the state buffers ping-pong):
 * ask again before every exchange, and order the writes before the next sweep on its stream.  After writing owned
 * planes through it, primitive fields written earlier are stale (halo planes: nobody reads theirs). */
int shasta_plane_ptr(shasta_t* h, int field, int z0, void** ptr_dev);
/* From now on the x and y sweeps update the planes z_lo .. z_hi-1 only (default: all, 0 .. nz); the z sweeps and the
 * element-wise passes still cover every plane.  For a z-slab rank: its halo planes are overwritten before each z sweep
 * anyway, so sweeping them along x and y is wasted work (8 of 8 + nz/P planes).  After an x or y sweep the planes
 * outside the range hold stale data (and stale primitives) until they are written again (shasta_set_planes, a z sweep).
 * 0 <= z_lo < z_hi <= nz, SHASTA_EINVAL otherwise; SHASTA_ESTATE with SHASTA_BATCH > 1. */
int shasta_set_active_planes(shasta_t* h, int z_lo, int z_hi);

/*
 * Advance nsteps time steps dt = lambda*dx.  One step = three fused sweep kernels, one per axis in
 * table order (axes of extent 1 are skipped); each sweep does, per pencil, in one pass over the five
 * conserved fields: ghost extension (boundary), cons2prim, half-step predictor transport (eq. (17) with
 * lambda/2), cons2prim, full-step transport with diffusion (eqs. (15)-(17)), phoenical antidiffusion with
 * the flux limiter (eqs. (18)-(22)), the causality projection, and -- in the last
 * sweep of a step -- cons2prim of the new state into the primitive fields.  Asynchronous on `stream`.
 */
int shasta_step(shasta_t* h, int nsteps, void* stream);

/* One sweep ("round") along `axis` (0=x,1=y,2=z) by the full dt: the fused kernel of
 * shasta_step, launched once.  emit_primitives: 0 = conserved fields only; 1 = also write the primitive fields of
 * the new state (as the last sweep of a step does); 2 = also write the primitive fields of the state BEFORE this
 * sweep (y and z only, SHASTA_EINVAL otherwise): what shasta_step uses after a step that ended with an x sweep.
 * Does not advance the step counter.  An axis of extent 1 is a no-op (reading G15).  Used by tests (single-axis
 * parity) and by bench.py to time each kernel with CUDA events. */
int shasta_sweep(shasta_t* h, int axis, int emit_primitives, void* stream);

/* Primitive fields of the current state (phases 3-4): e = E - |M| v,
 * n = R sqrt(1-v^2), p = EOS(e,n), v = root of v (E + p) = |M|.  Any pointer may be NULL = skip. */
int shasta_get_primitives(shasta_t* h, double* e_dev, double* p_dev, double* n_dev, double* vx_dev,
                          double* vy_dev, double* vz_dev, void* stream);
int shasta_get_primitives_host(shasta_t* h, double* e_host, double* p_host, double* n_host,
                               double* vx_host, double* vy_host, double* vz_host, void* stream);

/* dx^3 * sum over cells of E, Mx, My, Mz, R (the conserved totals of eqs. (12)-(14)),
 * compensated fp64 summation.  `totals_host` is a host pointer to 5 doubles (5*B for a batch of B events, event
 * after event).  SYNCHRONISES `stream`. */
int shasta_conserved_totals(shasta_t* h, double* totals_host, void* stream);

/* Cumulative counters since create (host pointer to 4 values): [0] cells where the projection Pi
 * (|M| <= (1-1e-12) E) fired at the end of a sweep, [1] vacuum cells (E <= 0) seen there,
 * [2] e < 0 floored, [3] p < 0 floored in the primitive output.  SYNCHRONISES the device. */
int shasta_diagnostics(shasta_t* h, unsigned long long* counts_host);

/* Number of kernels this handle has launched since create (bench.py's gpu_launches). */
long long shasta_launch_count(const shasta_t* h);
/* Number of CUDA-graph launches shasta_step has made (each replays one cycle of the axis table; SHASTA_GRAPH). */
long long shasta_graph_launch_count(const shasta_t* h);
/* Step counter s (number of steps taken, or the value set by SHASTA_STEP_INDEX). */
long long shasta_step_index(const shasta_t* h);
/* Name of the sweep kernel variant used for `axis` with the current options (for profiles/); the suffix "(cp.async)"
 * says that the sweep fills its shared-memory tiles without TMA (no 16 B row strides, SHASTA_NO_TMA, ...). */
const char* shasta_kernel_name(const shasta_t* h, int axis);

const char* shasta_last_error(const shasta_t* h);   /* h may be NULL: error of the last failed create or handle-less
                                                       call (shasta_conserved_totals_static) on this thread */

/*
 * The conserved totals of eqs. (12)-(14) for callers that may not allocate: CUDA-graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc.  No handle; this call makes no cudaMalloc, cudaMallocHost, cudaFree
 * or allocating library call, and does not synchronise.
 *   ncell                 number of cells, 0 <= ncell <= shasta_conserved_totals_static_max_cells() = 2^26 = 67 108 864
 *                         (a 406^3 grid; 256^3 is 2^24).  Beyond that: SHASTA_EINVAL, nothing launched.
 *   E_dev .. R_dev        DEVICE pointers, ncell doubles each (the caller's; read only)
 *   dv                    cell volume dx^3
 *   totals_dev            DEVICE pointer to 5 doubles (the caller's): dv * sum of E, Mx, My, Mz, R, compensated fp64
 *                         summation; written asynchronously on `stream`
 * Scratch: the per-block partial sums (which shasta_conserved_totals keeps in memory its handle allocated) live in a
 * file-scope `static __device__` array of 320 KiB that every GPU loading libshasta.so holds until the process exits;
 * its address is looked up once per device, on the first call made with that device current (make that first call
 * outside stream capture).  All calls on a device share the array and it keeps the last call's contents; nothing in
 * it has to start at zero (every slot a call reads it has written before).  Calls that can overlap on the GPU --
 * different streams, or graph branches, without an ordering between them -- RACE on it: order them.  The pointers
 * must belong to the current device.  Errors are reported through shasta_last_error(NULL).
 */
int shasta_conserved_totals_static(long long ncell, const double* E_dev, const double* Mx_dev, const double* My_dev,
                                   const double* Mz_dev, const double* R_dev, double dv, double* totals_dev,
                                   void* stream);
long long shasta_conserved_totals_static_max_cells(void);

#ifdef __cplusplus
}
#endif
#endif /* SHASTA_H */
