// Internal declarations shared by the translation units of libnpfem_b200.so.
#pragma once

#include <cuda_runtime.h>

#include <cstdint>
#include <string>
#include <vector>

#include "../../include/npfem.h"
#include "host_setup.hpp"

namespace npfem {

// Number of state fields kept per bucket, each [cells][3][n_pad] of the compute type.
// F_XL: fp32 contexts only (null in fp64 contexts): low part of the positions.  The cell-local position of a vertex
//       is the unevaluated sum x + xl with |xl| <= ulp(x)/2 (two-float storage): the epilogue
//       adds d to it with a compensated sum, so the rounding of x_{n+1} = x_n + d to fp32 does not accumulate in the
//       state over the steps, and the local step evaluates grad E at x + (xl + d)
enum Field { F_X = 0, F_V, F_F, F_B, F_D, F_G, F_XL, F_COUNT };

// Device tables of the scheduled fp32 local step (local_schedule.hpp / local_sched.cu).
struct SchedDev {
  bool valid = false;
  int threads = 0, vstride = 0, tpt = 0, ttri = 0, maxv = 0, n_vslots = 0, n_tslots = 0, n_cslots = 0;
  int ttri_used = 0;           // quad schedule: number of quads (threads below it own one)
  const uint32_t *tri_words = nullptr;
  const float *tri_consts = nullptr;
  const uint32_t *vtx_words = nullptr;
  const float *vtx_coef = nullptr;
  double vol_lane_bound = 0;   // max over threads of sum_j |x0| 2A_t of the rest shape (6V partial per lane)
};

// Device tables of the multi-pass quad local step (quadmp_schedule.hpp / local_quadmp.cu)
struct QuadMpDev {
  bool valid = false;
  int passes = 0, nq = 0, maxv = 0, lstride = 0, n_vslots = 0, n_tslots = 0, n_cslots = 0;
  int list_len[4] = {0, 0, 0, 0};
  const uint32_t *quad_words = nullptr;
  const float *quad_consts = nullptr;
  const uint32_t *list_words = nullptr;
  const uint32_t *vtx_slot = nullptr;
  const float *vtx_coef = nullptr;
  double vol_lane_bound = 0;
};

// Per-context launch state of the kernels that opt in to more than 48 KB of dynamic shared memory: the attribute
// is per device and function, the occupancy depends on it, so both are cached per context and cell type (a
// process-wide static would be wrong for two devices in one process).
// Opt a kernel in to the largest dynamic shared-memory size the SM allows next to its static shared memory
// (227 KB per CTA in all).  Always the maximum, never the size of the launch at hand: the attribute belongs to the
// function on the device, and two cell types (or two contexts) sharing a kernel must not lower each other's limit.
template <typename K>
inline cudaError_t opt_in_max_dynamic_smem(K kernel) {
  cudaFuncAttributes fa;
  cudaError_t e = cudaFuncGetAttributes(&fa, kernel);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - int(fa.sharedSizeBytes));
}

struct KernelCache {
  size_t sched_smem = 0, quad_smem = 0;
  int sched_per_sm = 0, quad_per_sm = 0;
  int tc_smem = 0;
  bool generic_attr[2] = {false, false}, smem_attr = false, big_attr = false, fused_attr = false, objective_attr = false,
       damping_attr = false, quadmp_attr = false;
};

// Device view of one cell type (pointers into the workspace; element type = compute type).
struct TypeDev {
  int n = 0, T = 0, n_pad = 0, valence_max = 0;
  const int4 *tri = nullptr;         // [T]  v0 v1 v2 0
  const int4 *tri_nbr = nullptr;     // [T]  t0 t1 t2 0
  const void *tri_rest = nullptr;    // [T][4]  a b c A0
  const void *hinge_rest = nullptr;  // [T][6]  (cos, sin) theta0 per edge
  const int *vtx_corner = nullptr;   // [valence_max][n]
  const int *vtx_nbr = nullptr;      // [valence_max][n]
  const void *vtx_w = nullptr;       // [valence_max+1][n]
  const void *vtx_mass = nullptr;    // [n]  m_v
  const void *vtx_inv_area = nullptr;// [n]  1/A_v
  const void *Hinv = nullptr;        // [n_pad][n_pad] dense inverse of H~ (compute type)
  const void *Hinv_tf32 = nullptr;   // fp32 contexts: H~^-1 rounded to TF32 to nearest (the tensor-core operand W_hi)
  const void *Hinv_lo = nullptr;     // fp32 contexts: W_lo = tf32(H~^-1 - W_hi), the second term of the split operator
  // fp32 shared-memory local step (local_smem.cu)
  const void *tri_pack = nullptr;    // [T] uint4: v0|v1<<16, v2|n0<<16, n1|n2<<16, 0
  const void *vtx_pack = nullptr;    // [n] uint4: 8 x u16 corner ids (3T = none)
  const void *vtx_coef = nullptr;    // [n] float: (1 - gamma)(1 + h alpha) m_v / h^2
  double gamma = 0;                  // (beta/h) / (1 + beta/h)   // fp32 contexts: same, rounded to TF32, tiled for tcgen05 (may be null)
  // scalars (double; converted at launch)
  double h = 0, B4 = 0, C4 = 0, k_b = 0, kv_over_V0 = 0, V0 = 0, k_mem = 0, beta_over_h = 0;
  double inertia_coef = 0;           // (1 + h alpha) / h^2, multiplies m_v
  double kappa = 0;
  SchedDev sched;                    // fp32 contexts: scheduled local step (may be invalid)
  SchedDev quad;                     // fp32 contexts: quad local step (quad_schedule.hpp / local_quad.cu; may be invalid)
  QuadMpDev quadmp;                  // fp32 contexts, meshes beyond one pass: multi-pass quad local step (may be invalid)
  mutable KernelCache cache;
};

// One bucket = all cells of one type, contiguous slots.
struct Bucket {
  int type = 0;
  int64_t cells = 0;
  void *field[F_COUNT] = {};         // each [cells][3][n_pad]
  double *origin = nullptr;          // [cells][3] fp64 per-cell origin of the local coordinates
  double *objective = nullptr;       // [NPFEM_MAX_ITERATIONS+1][cells] (diagnostics; lazily allocated)
  void *scratch = nullptr;           // generic local step: per-CTA normals + corner forces when they do not fit smem
};

// Per listed cell: where its block sits in the user buffer and where it lives in the workspace.
struct CellRef {
  int64_t user_offset;   // element offset of the cell's [n][3] block in the user buffer
  int32_t bucket;
  int32_t slot;
};

// ---- launchers (each enqueues on `stream`, returns the number of kernels launched or <0) -------
// tmp: device scratch of invert_spd_tmp_doubles(n) doubles (from the workspace: the library allocates nothing here)
size_t invert_spd_tmp_doubles(int n);
int launch_invert_spd(const double *H_dev, double *Hinv_dev, int n, double *tmp, cudaStream_t stream,
                      double *residual_out, std::string &err);

int launch_convert_pad(const double *X, int n, void *out, int n_pad, int precision, cudaStream_t s);
// out = in rounded to TF32 to nearest (the tensor core would otherwise drop the low 13 mantissa bits)
int launch_round_tf32(const float *in, float *out, size_t count, cudaStream_t s);

// implemented per operation in pack.cu
struct PackArgs {
  const CellRef *refs;     // device
  int64_t n_refs;
  const void *src_a;       // positions / forces (device, io dtype) or nullptr
  const void *src_b;       // velocities or nullptr
  void *dst_a;             // get_state outputs
  void *dst_b;
  int io_dtype;
};

// The TF32 tensor-core path reads fp32 operands and IGNORES their low 13 mantissa bits (truncation).  Truncating both
// operands biases every product towards zero and costs 1.3e-3 of the net momentum of a cell;
// rounding them to nearest beforehand leaves 3e-6.  Both operands are therefore stored already rounded.
__device__ __forceinline__ float tf32_rn(float x) {
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
  return __uint_as_float(r);
}
__device__ __forceinline__ double tf32_rn(double x) { return x; }   // fp64 contexts never take the TF32 path

struct BucketView {       // what kernels need of a bucket, passed by value
  void *field[F_COUNT];
  double *origin;
  int64_t cells;
  int n, n_pad;
  int g_tf32;              // the local step rounds g to TF32 (to nearest): its consumer is the TF32 tensor-core GEMM
};

int launch_set_state(const BucketView *views_dev, const PackArgs &a, int precision, cudaStream_t s);
int launch_set_forces(const BucketView *views_dev, const PackArgs &a, int precision, cudaStream_t s);
int launch_get_state(const BucketView *views_dev, const PackArgs &a, int precision, cudaStream_t s);

int launch_prologue(const TypeDev &td, const BucketView &bv, int precision, cudaStream_t s);
int launch_epilogue(const TypeDev &td, const BucketView &bv, int precision, double v_max, cudaStream_t s);

// PIK collision term (coupling.cu): per bucket, targets [cells][3][n_pad] in GLOBAL coordinates, fp64 (the origin of
// a cell's local frame moves when the prologue re-centres it or set_state is called again; global targets stay
// valid), and stiffness [cells][n_pad] (0 = vertex not in contact), compute type
struct CollisionDev {
  double *targets = nullptr;
  void *stiffness = nullptr;
};
int launch_set_collisions(const BucketView *views_dev, const CollisionDev *cols_dev, const PackArgs &a, int precision,
                          cudaStream_t s);   // a.src_a = targets, a.src_b = stiffness
int launch_collision_grad(const BucketView &bv, const CollisionDev &col, int precision, cudaStream_t s);
int launch_collision_energy(const BucketView &bv, const CollisionDev &col, const int64_t *cell_id_dev, double *out,
                            const int *skip_dev, int precision, cudaStream_t s);

// one-ring median filter of the forces of the listed cells that belong to `bucket` (coupling.cu)
int launch_median_filter(const BucketView *views_dev, const CellRef *refs_dev, int64_t n_refs, int bucket,
                         const TypeDev &td, int precision, cudaStream_t s);

// local step: g = M~ d/h^2 - b + grad E(x_n + d)
size_t local_generic_scratch_bytes(const TypeDev &td, int precision, int n_sm);
int launch_local_generic(const TypeDev &td, const BucketView &bv, void *scratch, int precision, int n_sm,
                         cudaStream_t s);
// cell_id_dev == nullptr: objective_row is indexed by the bucket slot; skip_dev[slot] != 0 skips a cell
int launch_objective(const TypeDev &td, const BucketView &bv, const int64_t *cell_id_dev, double *objective_row,
                     const int *skip_dev, int precision, int n_sm, cudaStream_t s);

// Armijo backtracking line search, per-cell state of one bucket
struct LineSearchDev {
  double *obj0 = nullptr, *obj1 = nullptr, *slope = nullptr, *alpha = nullptr;   // [cells]
  int *done = nullptr;   // [cells + 1]: 1 = step length settled; done[cells] = number of cells still searching (kernels
                         // that are given `done` as their skip list return at once when it is 0)
  void *d_old = nullptr;                                                          // [cells][3][n_pad] d before the global step
  // fp32 contexts whose global step runs on the TF32 tensor cores: the search direction comes from a 3xTF32
  // product (g = g_hi + g_lo, H~^-1 = W_hi + W_lo, the lo x lo term dropped), see launch_ls_split_g
  float *g_lo = nullptr;                                                          // [cells][3][n_pad]
};
// g <- tf32(g), g_lo <- tf32(g - tf32(g)) over count elements; w_lo <- tf32(w - w_hi)
int launch_ls_split_g(float *g, float *g_lo, size_t count, cudaStream_t s);
int launch_ls_split_w(const float *w, const float *w_hi, float *w_lo, size_t count, cudaStream_t s);
// fp32: g (reduced gradient of a fast local-step kernel) += gamma m^ d + (beta/h) L z -> the full gradient;
// rounds to TF32 when bv.g_tf32.  Returns -1 when the cell does not fit shared memory.
// g_lo != nullptr: also leaves the 3xTF32 split g = tf32(grad), g_lo = tf32(grad - g) (launch_ls_split_g)
int launch_damping_grad(const TypeDev &td, const BucketView &bv, float *g_lo, int n_sm, cudaStream_t s);
// after the global step: d holds d_old + p, u holds d_old, g the gradient.  slope = <g, p>, alpha = 1,
// done = frozen (||g|| <= grad_tol ||b||: alpha = 0, d restored); g is overwritten with p
int launch_ls_init(const BucketView &bv, const LineSearchDev &ls, double grad_tol, int precision, cudaStream_t s);
// per cell not done: accept if obj1 <= obj0 + c1 alpha slope (or `last`), else alpha /= 2, d = d_old + alpha p
int launch_ls_accept(const BucketView &bv, const LineSearchDev &ls, double c1, bool last, int precision, cudaStream_t s);

// global step: d <- d - g Hinv   ([3 cells x n_pad] . [n_pad x n_pad])
int launch_global_simt(const TypeDev &td, const BucketView &bv, int precision, double d_scale, cudaStream_t s);
// fp32 contexts, TF32 tensor cores (tcgen05); returns -1 when the shape is unsupported
bool global_tcgen05_supported(const TypeDev &td);
// d <- d_scale d - g Hinv.  Returns -1 for an unsupported shape, -2 when the launch itself failed (the CUDA error
// is left for the caller's cudaGetLastError: a failed tensor-core launch is an error, never a silent SIMT fallback)
int launch_global_tcgen05(const TypeDev &td, const BucketView &bv, int n_sm, double d_scale,
                          cudaStream_t s, const void *g_lo = nullptr, const void *w_lo = nullptr);

// fp32 fast local step; writes the reduced gradient (global step must then use d_scale = 1 - gamma)
bool local_smem_supported(const TypeDev &td);
int launch_local_smem(const TypeDev &td, const BucketView &bv, int n_sm, cudaStream_t s);

// fp32 scheduled local step (register-resident topology, conflict-free shared-memory slots); same
// reduced-gradient convention as launch_local_smem
bool local_sched_supported(const TypeDev &td);
int launch_local_sched(const TypeDev &td, const BucketView &bv, int n_sm, cudaStream_t s);

// fp32 quad local step: one thread per pair of adjacent triangles; same reduced-gradient convention
bool local_quad_supported(const TypeDev &td);
int launch_local_quad(const TypeDev &td, const BucketView &bv, int n_sm, cudaStream_t s);
// the same for meshes of up to 4 x 640 quads (RBC-2562): the quads in passes, per-vertex accumulators in shared memory
bool local_quadmp_supported(const TypeDev &td);
int launch_local_quadmp(const TypeDev &td, const BucketView &bv, int n_sm, cudaStream_t s);

// fp32 reduced-gradient local step for types too large for the scheduled kernel (chunked corner forces)
bool local_big_supported(const TypeDev &td);
int launch_local_big(const TypeDev &td, const BucketView &bv, int n_sm, cudaStream_t s);

// whole time step of a cell in one kernel (small batches; step_fused.cu)
bool step_fused_supported(const TypeDev &td);
int launch_step_fused(const TypeDev &td, const BucketView &bv, int n_sm, int n_iterations, double v_max, cudaStream_t s);

int launch_monotone_flags(const double *history, int n_entries, int64_t cells, int32_t *flags, cudaStream_t s);

}  // namespace npfem
