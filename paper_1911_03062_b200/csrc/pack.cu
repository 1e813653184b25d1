// Boundary kernels: user buffers (the paper's x in R^{n x 3}, `[n][3]` per cell)
// <-> the batched structure-of-arrays state `field[cell][3][n_pad]` in cell-local coordinates.
//
// Local coordinates: each cell keeps an fp64 origin (its centroid at set_state time); the stored
// positions are x - origin in the compute type, so fp32 contexts keep full relative precision for
// cells placed hundreds of micrometres from the domain origin ("fp32 state").
#include "internal.h"

namespace npfem {
namespace {

template <typename U>
__device__ __forceinline__ double load_as_double(const void *p, int64_t i) {
  return double(reinterpret_cast<const U *>(p)[i]);
}

__device__ __forceinline__ double block_sum(double v, double *red) {
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  const int w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  __syncthreads();
  if ((threadIdx.x & 31) == 0) red[w] = v;
  __syncthreads();
  double s = 0.0;
  for (int i = 0; i < nw; ++i) s += red[i];
  return s;
}

// one CTA per listed cell
template <typename T, typename U>
__global__ void __launch_bounds__(256)
set_state_kernel(const BucketView *__restrict__ views, const CellRef *__restrict__ refs,
                 const void *__restrict__ pos, const void *__restrict__ vel) {
  __shared__ double red[8];
  const CellRef ref = refs[blockIdx.x];
  const BucketView bv = views[ref.bucket];
  const int n = bv.n, n_pad = bv.n_pad;
  const size_t base = size_t(ref.slot) * 3 * n_pad;
  double c[3] = {0.0, 0.0, 0.0};
  for (int i = threadIdx.x; i < 3 * n; i += blockDim.x) c[i % 3] += load_as_double<U>(pos, ref.user_offset + i);
  double origin[3];
  for (int k = 0; k < 3; ++k) origin[k] = block_sum(c[k], red) / n;
  if (threadIdx.x < 3) bv.origin[size_t(ref.slot) * 3 + threadIdx.x] = origin[threadIdx.x];
  T *x = static_cast<T *>(bv.field[F_X]) + base;
  T *v = static_cast<T *>(bv.field[F_V]) + base;
  T *xl = bv.field[F_XL] ? static_cast<T *>(bv.field[F_XL]) + base : nullptr;   // fp32 contexts: two-float positions
  for (int i = threadIdx.x; i < 3 * n; i += blockDim.x) {
    const int vert = i / 3, k = i % 3;
    const double local = load_as_double<U>(pos, ref.user_offset + i) - origin[k];
    const T hi = T(local);
    x[k * n_pad + vert] = hi;
    if (xl) xl[k * n_pad + vert] = T(local - double(hi));
    v[k * n_pad + vert] = vel ? T(load_as_double<U>(vel, ref.user_offset + i)) : T(0);
  }
  // forces, rhs, displacement, gradient start at zero; padding columns of every field are zero
  for (int f = 0; f < F_COUNT; ++f) {
    if (!bv.field[f]) continue;
    T *p = static_cast<T *>(bv.field[f]) + base;
    const bool whole = (f != F_X && f != F_V && f != F_XL);
    for (int i = threadIdx.x; i < 3 * n_pad; i += blockDim.x)
      if (whole || (i % n_pad) >= n) p[i] = T(0);
  }
}

template <typename T, typename U>
__global__ void __launch_bounds__(256)
set_forces_kernel(const BucketView *__restrict__ views, const CellRef *__restrict__ refs,
                  const void *__restrict__ frc) {
  const CellRef ref = refs[blockIdx.x];
  const BucketView bv = views[ref.bucket];
  const int n = bv.n, n_pad = bv.n_pad;
  T *f = static_cast<T *>(bv.field[F_F]) + size_t(ref.slot) * 3 * n_pad;
  for (int i = threadIdx.x; i < 3 * n; i += blockDim.x)
    f[(i % 3) * n_pad + i / 3] = T(load_as_double<U>(frc, ref.user_offset + i));
}

template <typename T, typename U>
__global__ void __launch_bounds__(256)
get_state_kernel(const BucketView *__restrict__ views, const CellRef *__restrict__ refs,
                 void *__restrict__ pos, void *__restrict__ vel) {
  const CellRef ref = refs[blockIdx.x];
  const BucketView bv = views[ref.bucket];
  const int n = bv.n, n_pad = bv.n_pad;
  const size_t base = size_t(ref.slot) * 3 * n_pad;
  const T *x = static_cast<const T *>(bv.field[F_X]) + base;
  const T *v = static_cast<const T *>(bv.field[F_V]) + base;
  const T *xl = bv.field[F_XL] ? static_cast<const T *>(bv.field[F_XL]) + base : nullptr;
  const double *origin = bv.origin + size_t(ref.slot) * 3;
  for (int i = threadIdx.x; i < 3 * n; i += blockDim.x) {
    const int vert = i / 3, k = i % 3;
    const double lo = xl ? double(xl[k * n_pad + vert]) : 0.0;
    if (pos) reinterpret_cast<U *>(pos)[ref.user_offset + i] = U(origin[k] + (double(x[k * n_pad + vert]) + lo));
    if (vel) reinterpret_cast<U *>(vel)[ref.user_offset + i] = U(v[k * n_pad + vert]);
  }
}

template <template <typename, typename> class Launcher, typename... Args>
int dispatch(int precision, int io_dtype, Args... args) {
  if (precision == NPFEM_F32 && io_dtype == NPFEM_F32) return Launcher<float, float>::run(args...);
  if (precision == NPFEM_F32 && io_dtype == NPFEM_F64) return Launcher<float, double>::run(args...);
  if (precision == NPFEM_F64 && io_dtype == NPFEM_F32) return Launcher<double, float>::run(args...);
  return Launcher<double, double>::run(args...);
}

template <typename T, typename U>
struct SetState {
  static int run(const BucketView *views, const PackArgs &a, cudaStream_t s) {
    set_state_kernel<T, U><<<unsigned(a.n_refs), 256, 0, s>>>(views, a.refs, a.src_a, a.src_b);
    return 1;
  }
};
template <typename T, typename U>
struct SetForces {
  static int run(const BucketView *views, const PackArgs &a, cudaStream_t s) {
    set_forces_kernel<T, U><<<unsigned(a.n_refs), 256, 0, s>>>(views, a.refs, a.src_a);
    return 1;
  }
};
template <typename T, typename U>
struct GetState {
  static int run(const BucketView *views, const PackArgs &a, cudaStream_t s) {
    get_state_kernel<T, U><<<unsigned(a.n_refs), 256, 0, s>>>(views, a.refs, a.dst_a, a.dst_b);
    return 1;
  }
};

}  // namespace

int launch_set_state(const BucketView *views_dev, const PackArgs &a, int precision, cudaStream_t s) {
  if (a.n_refs == 0) return 0;
  return dispatch<SetState>(precision, a.io_dtype, views_dev, a, s);
}
int launch_set_forces(const BucketView *views_dev, const PackArgs &a, int precision, cudaStream_t s) {
  if (a.n_refs == 0) return 0;
  return dispatch<SetForces>(precision, a.io_dtype, views_dev, a, s);
}
int launch_get_state(const BucketView *views_dev, const PackArgs &a, int precision, cudaStream_t s) {
  if (a.n_refs == 0) return 0;
  return dispatch<GetState>(precision, a.io_dtype, views_dev, a, s);
}

// diagnostics: flags[c] = 1 if history[k+1][c] <= history[k][c] (within round-off) for all k
__global__ void monotone_kernel(const double *__restrict__ hist, int n_entries, int64_t cells,
                                int32_t *__restrict__ flags) {
  const int64_t c = blockIdx.x * int64_t(blockDim.x) + threadIdx.x;
  if (c >= cells) return;
  int ok = 1;
  for (int k = 0; k + 1 < n_entries; ++k) {
    const double a = hist[size_t(k) * cells + c], b = hist[size_t(k + 1) * cells + c];
    if (b > a + 1e-12 * (fabs(a) + fabs(b))) ok = 0;
  }
  flags[c] = ok;
}

int launch_monotone_flags(const double *history, int n_entries, int64_t cells, int32_t *flags, cudaStream_t s) {
  if (cells == 0) return 0;
  monotone_kernel<<<unsigned((cells + 255) / 256), 256, 0, s>>>(history, n_entries, cells, flags);
  return 1;
}

}  // namespace npfem
