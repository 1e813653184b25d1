// Per-cell Armijo backtracking line search and gradient-norm stopping test.
//
// The paper's text has no line search (reading R2: step length 1) but claims "unconditional
// stability for arbitrary time steps"; with large steps / forces the plain
// iteration of Eq. (4) diverges.  Per cell and iteration, with grad = grad g(d), p = -H~^-1 grad:
//   frozen if ||grad||_2 <= grad_tol ||b||_2 (alpha = 0);  otherwise alpha = 1 and alpha is halved while
//   g(d + alpha p) > g(d) + c1 alpha <grad, p>, at most max_halvings times;  d <- d + alpha p.
// npfem_step drives it (api.cu): local step (full gradient) -> objective g(d) (first iteration of a step
// only: afterwards it is the objective of the accepted trial point) -> d_old := d ->
// global step (d := d_old + p) -> ls_init -> (max_halvings + 1) x [objective at the trial point ->
// ls_accept].  All decisions are taken in fp64 on per-cell fp64 reductions; one warp per cell.
#include "internal.h"

namespace npfem {
namespace {

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

template <typename T>
__global__ void __launch_bounds__(128)
ls_init_kernel(BucketView bv, LineSearchDev ls, double grad_tol) {
  const int lane = threadIdx.x & 31;
  const int64_t warp0 = (int64_t(blockIdx.x) * blockDim.x + threadIdx.x) >> 5;
  const int64_t n_warps = (int64_t(gridDim.x) * blockDim.x) >> 5;
  const int n = bv.n, n_pad = bv.n_pad;
  for (int64_t cell = warp0; cell < bv.cells; cell += n_warps) {
    const size_t base = size_t(cell) * 3 * n_pad;
    T *g = static_cast<T *>(bv.field[F_G]) + base;
    T *d = static_cast<T *>(bv.field[F_D]) + base;
    const T *d_old = static_cast<const T *>(bv.field[F_U]) + base;
    const T *b = static_cast<const T *>(bv.field[F_B]) + base;
    double slope = 0.0, gg = 0.0, bb = 0.0;
    for (int k = 0; k < 3; ++k)
      for (int i = lane; i < n; i += 32) {
        const int o = k * n_pad + i;
        const T p = d[o] - d_old[o];            // the search direction, rounded once to the compute type
        const double gi = double(g[o]), bi = double(b[o]);
        slope += gi * double(p);
        gg += gi * gi;
        bb += bi * bi;
        g[o] = p;                               // the gradient is not needed any more: keep p in its place
      }
    slope = warp_sum(slope);
    gg = warp_sum(gg);
    bb = warp_sum(bb);
    const bool frozen = sqrt(gg) <= grad_tol * sqrt(bb);
    if (frozen)
      for (int k = 0; k < 3; ++k)
        for (int i = lane; i < n; i += 32) d[k * n_pad + i] = d_old[k * n_pad + i];
    if (lane == 0) {
      ls.slope[cell] = slope;
      ls.alpha[cell] = frozen ? 0.0 : 1.0;
      ls.done[cell] = frozen ? 1 : 0;
    }
  }
}

template <typename T>
__global__ void __launch_bounds__(128)
ls_accept_kernel(BucketView bv, LineSearchDev ls, double c1, int last) {
  const int lane = threadIdx.x & 31;
  const int64_t warp0 = (int64_t(blockIdx.x) * blockDim.x + threadIdx.x) >> 5;
  const int64_t n_warps = (int64_t(gridDim.x) * blockDim.x) >> 5;
  const int n = bv.n, n_pad = bv.n_pad;
  for (int64_t cell = warp0; cell < bv.cells; cell += n_warps) {
    if (ls.done[cell]) continue;                // warp-uniform
    const double alpha = ls.alpha[cell];
    const bool ok = ls.obj1[cell] <= ls.obj0[cell] + c1 * alpha * ls.slope[cell];
    __syncwarp();
    if (ok || last) {
      // d stays at this trial point, so its objective is g(d) of the next iteration of this step (api.cu
      // evaluates obj0 at the first iteration only); frozen cells never get here and keep theirs
      if (lane == 0) {
        ls.done[cell] = 1;
        ls.obj0[cell] = ls.obj1[cell];
      }
      continue;
    }
    const double half = 0.5 * alpha;
    const size_t base = size_t(cell) * 3 * n_pad;
    const T *p = static_cast<const T *>(bv.field[F_G]) + base;
    T *d = static_cast<T *>(bv.field[F_D]) + base;
    const T *d_old = static_cast<const T *>(bv.field[F_U]) + base;
    for (int k = 0; k < 3; ++k)
      for (int i = lane; i < n; i += 32) {
        const int o = k * n_pad + i;
        d[o] = d_old[o] + T(half) * p[o];       // alpha is a power of two: the product is exact
      }
    if (lane == 0) ls.alpha[cell] = half;
  }
}

unsigned warp_grid(int64_t cells) {
  const int64_t ctas = (cells + 3) / 4;
  return unsigned(ctas < 148 * 16 ? ctas : 148 * 16);
}

}  // namespace

int launch_ls_init(const BucketView &bv, const LineSearchDev &ls, double grad_tol, int precision, cudaStream_t s) {
  if (bv.cells == 0) return 0;
  if (precision == NPFEM_F32)
    ls_init_kernel<float><<<warp_grid(bv.cells), 128, 0, s>>>(bv, ls, grad_tol);
  else
    ls_init_kernel<double><<<warp_grid(bv.cells), 128, 0, s>>>(bv, ls, grad_tol);
  return 1;
}

int launch_ls_accept(const BucketView &bv, const LineSearchDev &ls, double c1, bool last, int precision, cudaStream_t s) {
  if (bv.cells == 0) return 0;
  if (precision == NPFEM_F32)
    ls_accept_kernel<float><<<warp_grid(bv.cells), 128, 0, s>>>(bv, ls, c1, last ? 1 : 0);
  else
    ls_accept_kernel<double><<<warp_grid(bv.cells), 128, 0, s>>>(bv, ls, c1, last ? 1 : 0);
  return 1;
}

}  // namespace npfem
