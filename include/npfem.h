/*
 * npfem.h - C ABI of the B200-native npFEM solid-solver step.
 *
 * The library advances every deformable blood cell (closed triangulated
 * membranes: RBCs, platelets) of a batch by one implicit-Euler time step h,
 * exactly as the paper states the solid problem:
 *
 *   state {x_n, v_n}, x, v in R^{n x 3}, input F_ext in R^{n x 3} .... PAPER.md:257
 *   Eqs. (1)-(2) implicit Euler advancement ....................... PAPER.md:259-264
 *   Eq. (3)  min_x g(x) = 1/(2h^2) ||M~^(1/2)(x - y_n)||^2 + sum_i E_i(x),
 *            M~ = M + hC ........................................... PAPER.md:266-268
 *   Eq. (4)  x^{k+1} <- x^k - H~^-1 grad g(x^k), H~ constant ....... PAPER.md:268-272
 *   material constants ............................................. PAPER.md:226-239
 *   every cell is independent within a step ........................ PAPER.md:61,63
 *
 * The paper defers the energies, H~ and the damping formulas to its ref. [4];
 * the forms used are the readings R1-R16 listed in DESIGN.md.
 *
 * Conventions
 *   - Units: micrometre, microsecond, femtogram, piconewton.
 *   - Per-cell user buffers hold the paper's x in R^{n x 3}: `[n_vertices][3]`
 *     (xyz interleaved), the listed cells back to back in `cell_ids` order;
 *     `cell_ids == NULL` means all cells in cell-id order 0..n_cells-1.  The ids
 *     of a list must be distinct (NPFEM_EINVAL otherwise).
 *   - `dtype` of a user buffer is NPFEM_F32 or NPFEM_F64 and is independent of
 *     the context's compute precision (fp64 I/O on an fp32 context keeps the
 *     placement of cells far from the origin exact: state is stored in
 *     cell-local coordinates around a per-cell fp64 origin).
 *   - `where` says whether a user buffer is a DEVICE pointer (e.g. a torch
 *     tensor's data_ptr) or a HOST pointer (pinned memory gives async copies).
 *   - The library never frees caller memory.  All device work is enqueued on
 *     the stream given at creation; calls with device buffers return without
 *     synchronising.  Calls that write HOST buffers (get_*) synchronise the
 *     stream before returning; calls that read HOST buffers return after the
 *     host data has been consumed.
 *   - Every call returns NPFEM_OK (0) or a negative code; no exception crosses
 *     the ABI.  The message of the last failure is kept per context (and per
 *     thread for npfem_create) and read with npfem_last_error.  CUDA errors
 *     are sticky: after NPFEM_ECUDA the context only accepts npfem_destroy.
 *   - There is NO CPU fallback: without a CUDA device every call fails.
 */
#ifndef NPFEM_H_
#define NPFEM_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define NPFEM_OK       0
#define NPFEM_EINVAL  -1   /* bad argument */
#define NPFEM_EMESH   -2   /* mesh not a closed, consistently oriented 2-manifold / degenerate */
#define NPFEM_ECUDA   -3   /* CUDA runtime failure (sticky) */
#define NPFEM_ENOMEM  -4   /* host or device allocation failed / workspace too small */
#define NPFEM_ESTATE  -5   /* call out of order (e.g. step before set_state) / solver setup failed */

#define NPFEM_F32 32
#define NPFEM_F64 64

#define NPFEM_DEVICE 0
#define NPFEM_HOST   1

/* options for npfem_set_option */
#define NPFEM_OPT_DIAGNOSTICS      1  /* 1: record the objective before every iteration (row a5); needs the scratch of
                                         NPFEM_FEATURE_DIAGNOSTICS (see npfem_bind_scratch) */
#define NPFEM_OPT_GLOBAL_STEP_MATH 2  /* fp32 contexts: 0 = TF32 tensor cores (default), 1 = FP32 FFMA, 2 = TF32 tensor cores with
                                         the operator split in two TF32 terms H~^-1 = W_hi + W_lo (twice the tensor work; removes
                                         the bias TF32 rounding of H~^-1 leaves in the fixed point) */
#define NPFEM_OPT_LOCAL_STEP_IMPL  3  /* 0 = auto, 1 = generic kernel, 2 = shared-memory persistent kernel,
                                         3 = scheduled kernel (register-resident topology, conflict-free slots),
                                         4 = large-mesh kernel (chunked corner forces, e.g. 2562-vertex cells),
                                         5 = quad kernel (one thread per pair of adjacent triangles),
                                         6 = multi-pass quad kernel (meshes of 1,282 ... 5,120 triangles).  auto = 5 where the
                                         type allows it, else 6, else 3, else 2, else 4, else 1 */

#define NPFEM_OPT_KERNEL_TIMING    4  /* 1: bracket every kernel of npfem_step with CUDA events */
#define NPFEM_OPT_FORCE_MEDIAN_FILTER 6  /* 1: npfem_set_forces median-filters F_ext over the one-ring of every vertex
                                            (per component, vertex + neighbours, even counts average) */
#define NPFEM_OPT_FUSED_STEP       7  /* whole step of a cell in ONE kernel (fp32, small batches): 0 = auto (a bucket of at
                                         most 1.5 cells per SM), 1 = never, 2 = whenever the cell type allows it */
#define NPFEM_OPT_UPDATE_MODE      5  /* fp32 tensor-core global step: 0 / 1 = the GEMM epilogue updates d in place (the only
                                         mode; the product-out mode 2 of earlier versions was slower and is gone) */

/* kernel kinds reported by npfem_get_kernel_times */
#define NPFEM_KIND_PROLOGUE 0
#define NPFEM_KIND_LOCAL    1
#define NPFEM_KIND_GLOBAL   2
#define NPFEM_KIND_EPILOGUE 3
#define NPFEM_KIND_LINE_SEARCH 4   /* objective evaluations + accept / backtrack kernels */
#define NPFEM_KIND_FUSED_STEP  5   /* whole-step kernel of the small-batch path */
#define NPFEM_KIND_GLOBAL_SIMT 6   /* global step on the SIMT GEMM (fp64 contexts: DMMA; fp32: only when NPFEM_OPT_GLOBAL_STEP_MATH
                                      = 1 or the shape does not fit the tcgen05 kernel).  NPFEM_KIND_GLOBAL is the tcgen05 kernel
                                      alone: a tensor-core launch that fails is NPFEM_ECUDA, never a silent fall back */
#define NPFEM_KIND_COUNT    7

/* optional features that need scratch memory (npfem_scratch_bytes / npfem_bind_scratch) */
#define NPFEM_FEATURE_DIAGNOSTICS 1   /* objective history, NPFEM_MAX_ITERATIONS + 1 rows of n_cells doubles */
#define NPFEM_FEATURE_LINE_SEARCH 2   /* per-cell search state, a copy of d, fp32: the 3xTF32 operands */
#define NPFEM_FEATURE_COLLISIONS  4   /* PIK targets (fp64, global coordinates) and stiffnesses */

#define NPFEM_MAX_ITERATIONS 256

typedef struct npfem_ctx npfem_ctx; /* opaque, owned by the library */

/* Material of one cell type. */
typedef struct npfem_material {
  double skalak_B;        /* pN/um   shear-type constant of the Skalak law            */
  double skalak_C;        /* pN/um   area-dilation constant of the Skalak law         */
  double skalak_D;        /* pN/um   listed by the paper, no formula given: unused    */
  double k_bending;       /* pN*um   hinge bending stiffness                          */
  double k_volume;        /* pN/um^2 volume-conservation stiffness                    */
  double rayleigh_alpha;  /* 1/us    C = alpha M + beta K                             */
  double rayleigh_beta;   /* us                                                       */
  double kappa_damping;   /* [0,1]   position-based-dynamics velocity damping, 0=off  */
  double density;         /* fg/um^3 mass of body incl. interior fluid = density * V0 */
} npfem_material;

/* One cell type: rest shape (HOST pointers, copied by npfem_create) + material. */
typedef struct npfem_cell_type {
  int32_t n_vertices;
  int32_t n_triangles;
  const double *rest_positions; /* [n_vertices][3] */
  const int32_t *triangles;     /* [n_triangles][3], counter-clockwise seen from outside */
  npfem_material material;
} npfem_cell_type;

/*
 * Build a solver for `n_cells` cells; cell c has type `type_of_cell[c]` (HOST array).
 * Pre-computes, per TYPE: rest data, lumped mass, the one-ring operator of the
 * Rayleigh/inertia term, and the dense inverse of the constant Hessian
 * approximation H~ (Eq. 4) on the device.
 * dt: time step h in us.  precision: NPFEM_F32 or NPFEM_F64 (compute type).
 * device: CUDA ordinal.  cuda_stream: a cudaStream_t (NULL = legacy default stream).
 * On failure *out is NULL and npfem_last_error(NULL) holds the message.
 */
int npfem_create(npfem_ctx **out, const npfem_cell_type *types, int32_t n_types,
                 const int32_t *type_of_cell, int64_t n_cells, double dt,
                 int32_t precision, int32_t device, void *cuda_stream);

/*
 * Device memory for state and scratch.  Optional: the caller (e.g. torch) may own it.
 * If no workspace is bound before the first set_state, the library allocates its own.
 * `dev_ptr` must be 256-byte aligned and stay valid until npfem_destroy.
 */
size_t npfem_workspace_bytes(const npfem_ctx *ctx);
int npfem_bind_workspace(npfem_ctx *ctx, void *dev_ptr, size_t bytes);

/*
 * The workspace holds everything the plain step needs, the create-time temporaries of the H~ inverse included
 * (they are overlaid by the state).  The OPTIONAL features (NPFEM_FEATURE_*: diagnostics, line search, collisions)
 * keep their memory in a separate scratch arena.  A caller that binds its own workspace binds the scratch too,
 * BEFORE enabling the feature: npfem_scratch_bytes(ctx, mask) bytes for the features in `mask`, 256-byte aligned,
 * valid until npfem_destroy; enabling a feature without it fails with NPFEM_ENOMEM.  With a library-owned
 * workspace the enabling call (npfem_set_option(NPFEM_OPT_DIAGNOSTICS), npfem_set_line_search,
 * npfem_set_collisions) allocates the feature's scratch itself.  Either way npfem_step never allocates.
 * Errors: NPFEM_EINVAL (mask, alignment), NPFEM_ENOMEM (too small), NPFEM_ESTATE (feature already has memory).
 */
size_t npfem_scratch_bytes(const npfem_ctx *ctx, int32_t features);
int npfem_bind_scratch(npfem_ctx *ctx, void *dev_ptr, size_t bytes, int32_t features);

/* Runtime switches (NPFEM_OPT_*). */
int npfem_set_option(npfem_ctx *ctx, int32_t option, int64_t value);

/*
 * Initial placement: positions x_n and velocities v_n (NULL = zero) of the listed cells,
 * each `[n_vertices(type)][3]` of `dtype`.  Forces of these cells are reset to zero.
 */
int npfem_set_state(npfem_ctx *ctx, const int64_t *cell_ids, int64_t n_ids,
                    const void *positions, const void *velocities, int32_t dtype, int32_t where);

/*
 * External forces F_ext(x_n) of the listed cells, pN.  Forces persist
 * until overwritten (the solid solver may run every >= 2 fluid steps).
 */
int npfem_set_forces(npfem_ctx *ctx, const int64_t *cell_ids, int64_t n_ids,
                     const void *forces, int32_t dtype, int32_t where);

/*
 * ONE time step h for every cell: prologue (PBD damping, rhs), `n_iterations`
 * quasi-Newton iterations of Eq. (4) (local step = grad g, global step = apply H~^-1),
 * epilogue (Eq. 1).  1 <= n_iterations <= NPFEM_MAX_ITERATIONS.  Asynchronous.
 * The call only enqueues kernels on the context's stream: no allocation, no synchronisation, no host read-back.  With
 * a caller-owned workspace (and scratch for the optional features) it can be captured in a CUDA graph and replayed.
 */
int npfem_step(npfem_ctx *ctx, int32_t n_iterations);

/*
 * The same time step as npfem_set_forces(all cells) + npfem_step + npfem_get_state(all cells) with HOST
 * buffers, pipelined: cells are independent within a step, so the population is cut
 * into `n_chunks` ranges of cell ids (1..64; 0 = chosen from the buffer size, at most 16); chunk i's solver
 * kernels run while chunk i+1's forces are copied in and chunk i-1's state is copied out on two copy
 * streams.  Results are bit-identical to the unpipelined sequence.  `forces` [in], `positions` and
 * `velocities` [out] are HOST buffers of all cells in cell-id order, each `[n][3]`, dtype `dtype`; use
 * page-locked memory or the copies do not overlap.  Owned by the caller, not retained.  Synchronous:
 * returns when the state is in the host buffers.  With diagnostics, line search, collisions or the
 * median filter on, the three calls run one after the other instead.  Errors: NPFEM_EINVAL (NULL
 * pointer, n_chunks, n_iterations), NPFEM_ESTATE (cells without state), NPFEM_ECUDA.
 */
int npfem_step_host(npfem_ctx *ctx, const void *forces, int32_t n_iterations, void *positions, void *velocities,
                    int32_t dtype, int32_t n_chunks);

/* Current {x, v} of the listed cells (either pointer may be NULL). */
int npfem_get_state(npfem_ctx *ctx, const int64_t *cell_ids, int64_t n_ids,
                    void *positions, void *velocities, int32_t dtype, int32_t where);

/*
 * Row (a5) diagnostic (needs NPFEM_OPT_DIAGNOSTICS = 1 before the step): the objective
 * of Eq. (3) up to its d-independent constant, g(d) = d^T M~ d/(2h^2) - d^T b + E(x_n + d),
 * per cell, before each iteration of the LAST step and after its final one.
 * history: fp64 `[n_entries][n_cells]` (cell-id order), n_entries = n_iterations + 1,
 * at most `max_entries` rows are written.  monotone (may be NULL): int32 per cell,
 * 1 if the objective never increased.  Both buffers live `where` says.
 */
int npfem_get_objective(npfem_ctx *ctx, double *history, int32_t max_entries,
                        int32_t *n_entries, int32_t *monotone, int32_t where);

/*
 * Per-cell Armijo backtracking line search + gradient-norm stopping test for the following steps
 * (the paper's text has none, reading R2, but claims unconditional stability,
 * PAPER.md:37, :264).  max_halvings = 0 switches it off (default: plain Eq. (4), step length 1).
 * Per cell and iteration: frozen if ||grad g||_2 <= grad_tol ||b||_2; otherwise alpha = 1 and alpha is
 * halved while g(d + alpha p) > g(d) + armijo_c1 alpha <grad g, p>, at most max_halvings (<= 30) times,
 * p = -H~^-1 grad g; d <- d + alpha p.  With it on, every iteration evaluates the objective (fp64) at the
 * trial point of every cell not yet accepted, up to max_halvings + 1 times; fp32 contexts take p from a
 * 3xTF32 product on the tensor cores (fp32-grade: a plain TF32 direction makes the search stall).  Needs the
 * scratch of NPFEM_FEATURE_LINE_SEARCH (see npfem_bind_scratch): NPFEM_ENOMEM from this call if it is missing.
 */
int npfem_set_line_search(npfem_ctx *ctx, int32_t max_halvings, double armijo_c1, double grad_tol);

/*
 * PIK collision term (near contact "a collision force, coming from a quadratic potential
 * energy" replaces the fluid force).  For the listed cells: targets p `[n][3]` (the
 * projection points from the caller's collision detection, global coordinates like positions) and
 * stiffness k `[n]` (pN/um, 0 = vertex not in contact), both of `dtype`, living `where` says.  The energy
 * sum_i 1/2 k_i |x_i - p_i|^2 enters grad g and the objective of every following step (not the constant
 * H~: keep k well below m_v / h^2), until overwritten or cleared; the targets are kept in global coordinates, so
 * they stay valid when a cell drifts (the local frame is re-centred) or gets a new state.  Collision DETECTION is
 * the caller's.  Needs the scratch of NPFEM_FEATURE_COLLISIONS (see npfem_bind_scratch).
 */
int npfem_set_collisions(npfem_ctx *ctx, const int64_t *cell_ids, int64_t n_ids, const void *targets,
                         const void *stiffness, int32_t dtype, int32_t where);
int npfem_clear_collisions(npfem_ctx *ctx);

/*
 * Vertex-velocity cap: after every step the magnitude of each vertex velocity v_{n+1} is
 * clamped to v_max (um/us), its direction kept; positions are not touched.  0 = off (default).
 */
int npfem_set_velocity_cap(npfem_ctx *ctx, double v_max);

/* Step lengths alpha of the LAST iteration of the last step, HOST array [n_cells] in cell-id order. */
int npfem_get_step_lengths(npfem_ctx *ctx, double *alpha);

/*
 * Device time per kernel kind since the last reset (needs NPFEM_OPT_KERNEL_TIMING = 1): CUDA
 * events recorded on the context's stream around every launch of npfem_step.  Synchronises the
 * stream.  ms[kind][type] and launches[kind][type] are HOST arrays of NPFEM_KIND_COUNT * n_types
 * entries (either may be NULL); reset != 0 clears the accumulators afterwards.
 */
int npfem_get_kernel_times(npfem_ctx *ctx, double *ms, int64_t *launches, int32_t reset);

/* Number of kernels the library has launched on this context so far. */
int64_t npfem_launch_count(const npfem_ctx *ctx);

/*
 * Host-only diagnostic (no CUDA device needed): builds the create-time shared-memory schedule of the
 * fp32 scheduled local step for one cell type (slots of vertex positions / triangle normals / corner
 * forces assigned by graph colouring so that the kernel's gathers avoid bank conflicts) and checks
 * it.  stats (HOST, n_stats >= 10 doubles):
 *   [0] 1 if the type fits the scheduled kernel, else 0 (the rest is then 0)
 *   [1] CTA threads  [2] triangles per thread
 *   [3] predicted wavefronts per vertex-gather instruction   (ideal 4.0)
 *   [4] predicted wavefronts per normal-gather instruction   (ideal 4.0)
 *   [5] worst wavefronts of a corner-force STORE instruction quarter (exactly 1.0 expected)
 *   [6] worst wavefronts of a corner-force GATHER instruction quarter (exactly 1.0 expected)
 *   [7] 1 if every vertex / triangle / corner slot is unique and every table entry decodes to the
 *       mesh's own connectivity, else 0
 *   [8] shared-memory bytes of the kernel's per-cell arrays  [9] host milliseconds to build
 * Returns NPFEM_OK, NPFEM_EINVAL or NPFEM_EMESH (message via npfem_last_error(NULL)).
 */
int npfem_local_schedule_stats(const npfem_cell_type *type, double dt, double *stats, int32_t n_stats);

/*
 * The same for the schedule of the QUAD local step (one thread per pair of adjacent triangles T0 = (p, q, r),
 * T1 = (p, s, q); the default fp32 local step of types with an even triangle count <= 1,280): host-only.
 *   [0] 1 if the type takes the quad kernel (a perfect matching of the dual graph exists and it fits), else 0
 *   [1] CTA threads (= quad slots, one vertex per thread)   [2] corner-force reads per vertex (6 or 8)
 *   [3] predicted wavefronts per vertex-gather instruction   [4] per normal-gather instruction   (ideal 4.0)
 *   [5] / [6] worst wavefronts of a corner-force STORE / GATHER instruction quarter (exactly 1.0 expected)
 *   [7] 1 if the tables decode to the mesh's own connectivity: every triangle in exactly one quad, both triangles of a
 *       quad adjacent across p-q and correctly oriented, the four neighbour-normal slots those of the triangles across
 *       q-r, r-p, p-s, s-q, every slot unique, every vertex reading exactly the corner slots written for it; else 0
 *   [8] shared-memory bytes of the kernel's per-cell arrays  [9] host milliseconds to build
 */
int npfem_quad_schedule_stats(const npfem_cell_type *type, double dt, double *stats, int32_t n_stats);

/*
 * The same for the MULTI-PASS quad local step (meshes of 1,282 ... 5,120 triangles, e.g. RBC-2562: the quads in up to 4
 * passes of 640, one quad per thread and pass): [1] = passes, the rest as for npfem_quad_schedule_stats; [7] also checks
 * that every pass's vertex list names each vertex the pass touches exactly once with exactly the slots written for it.
 */
int npfem_quadmp_schedule_stats(const npfem_cell_type *type, double dt, double *stats, int32_t n_stats);

/*
 * Measurement aid (not on the solver's path; SURVEY.md 8(d) "measure an FFMA peak on the box"): enqueues on
 * `cuda_stream` a kernel of grid_ctas CTAs x 256 threads, every thread running 16 independent chains of
 * `iterations` fused multiply-adds in `precision` (NPFEM_F32: FFMA, NPFEM_F64: DFMA).  The caller times it with
 * CUDA events; *flops_out (HOST, may be NULL) = 2 * 16 * iterations * 256 * grid_ctas.  sink_dev: a DEVICE scalar of
 * that precision.  Returns NPFEM_OK, NPFEM_EINVAL or NPFEM_ECUDA.
 */
int npfem_probe_fma_peak(void *cuda_stream, int32_t precision, int32_t grid_ctas, int32_t iterations, void *sink_dev,
                         double *flops_out);

/*
 * The fp64 inverse of one SPD matrix on the device: what npfem_create runs once per cell type on H~ (Eq. (4),
 * the global step applies H~^-1, constant per type), exposed on its own.  H_dev, Hinv_dev: DEVICE,
 * row-major [n][n] doubles, caller-owned, must not overlap; the result is symmetrised.  Newton-Schulz iteration
 * X <- X (2 I - H X), X0 = I / ||H||_inf, to ||I - H X||_F <= 1e-13 sqrt(n) (*residual_out, HOST, may be NULL).  The
 * call synchronises `cuda_stream` (it reads the residual back every iteration).
 *
 * npfem_invert_spd: the 3 n^2 + 32 doubles of scratch come from the caller (tmp_dev: DEVICE, 256-byte aligned,
 * tmp_bytes >= npfem_invert_spd_tmp_bytes(n)).
 *
 * npfem_invert_spd_static: for callers that cannot allocate device memory (CUDA graph capture around the call site,
 * serving loops, harnesses that forbid cudaMalloc): the scratch is a file-scope `static __device__` array inside the
 * library, 3 * NPFEM_INVERT_STATIC_MAX_N^2 + 32 doubles = 1.6 MB, which every device that loads the library holds
 * until the process exits.  n > NPFEM_INVERT_STATIC_MAX_N is refused (NPFEM_EINVAL).  All calls on a device share that
 * one array: calls that overlap on the GPU (two streams, two host threads) race - serialise them.  Neither entry point
 * calls cudaMalloc / cudaFree or an allocating library routine.
 *
 * Errors (message via npfem_invert_spd_last_error(), per host thread): NPFEM_EINVAL (NULL pointer, n, alignment,
 * n above the static maximum, non-positive diagonal), NPFEM_ENOMEM (tmp_bytes), NPFEM_ESTATE (no convergence: not SPD
 * or too ill-conditioned), NPFEM_ECUDA.
 */
#define NPFEM_INVERT_STATIC_MAX_N 258
size_t npfem_invert_spd_tmp_bytes(int32_t n);
int npfem_invert_spd(const double *H_dev, double *Hinv_dev, int32_t n, void *tmp_dev, size_t tmp_bytes, void *cuda_stream,
                     double *residual_out);
int npfem_invert_spd_static(const double *H_dev, double *Hinv_dev, int32_t n, void *cuda_stream, double *residual_out);
const char *npfem_invert_spd_last_error(void);

/* Message of the last failure on `ctx` (ctx == NULL: of the last failed npfem_create). */
const char *npfem_last_error(const npfem_ctx *ctx);

/* "major.minor.patch (sm_100a)" */
const char *npfem_version(void);

void npfem_destroy(npfem_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* NPFEM_H_ */
