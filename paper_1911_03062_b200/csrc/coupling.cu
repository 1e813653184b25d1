// The solver's inputs from the fluid coupling that live on the solid side:
//   * median filter of F_ext over the one-ring of every vertex (reading R18: per vertex and
//     Cartesian component, the median over the vertex and its one-ring neighbours; an even count
//     averages the two central values), applied by npfem_set_forces when
//     NPFEM_OPT_FORCE_MEDIAN_FILTER is on;
//   * the vertex-velocity cap (reading R17) lives in the step epilogue (prologue.cu);
//   * the PIK collision energy sum_i 1/2 k_i |x_i - p_i|^2 over the vertices the collision detection flagged
//     (reading R19: it enters grad g and the objective, not the constant H~):
//     npfem_set_collisions stores targets p (GLOBAL coordinates, fp64: the origin of a cell's local frame moves when
//     the prologue re-centres it or set_state is called again) and stiffnesses k per vertex, the
//     gradient term is added to the local step's output, the energy to the objective.
#include "internal.h"

namespace npfem {
namespace {

// one CTA per listed cell of bucket `bucket`: forces of the cell -> shared memory -> medians -> back
template <typename T>
__global__ void __launch_bounds__(256)
median_filter_kernel(const BucketView *__restrict__ views, const CellRef *__restrict__ refs, int bucket,
                     const int *__restrict__ vtx_nbr, int valence_max) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  T *sf = reinterpret_cast<T *>(smem_raw);           // [3][n]
  const CellRef ref = refs[blockIdx.x];
  if (ref.bucket != bucket) return;
  const BucketView bv = views[bucket];
  const int n = bv.n, n_pad = bv.n_pad;
  T *f = static_cast<T *>(bv.field[F_F]) + size_t(ref.slot) * 3 * n_pad;
  for (int i = threadIdx.x; i < 3 * n; i += blockDim.x) sf[i] = f[(i / n) * n_pad + i % n];
  __syncthreads();
  for (int v = threadIdx.x; v < n; v += blockDim.x) {
    int idx[33];
    int cnt = 0;
    idx[cnt++] = v;
    for (int q = 0; q < valence_max; ++q) {
      const int u = vtx_nbr[q * n + v];
      if (u != v) idx[cnt++] = u;                     // the table pads with the vertex itself
    }
    for (int k = 0; k < 3; ++k) {
      T vals[33];
      for (int i = 0; i < cnt; ++i) {                 // insertion sort of <= 33 values
        const T x = sf[k * n + idx[i]];
        int j = i;
        while (j > 0 && vals[j - 1] > x) {
          vals[j] = vals[j - 1];
          --j;
        }
        vals[j] = x;
      }
      f[k * n_pad + v] = (cnt & 1) ? vals[cnt / 2] : T(0.5) * (vals[cnt / 2 - 1] + vals[cnt / 2]);
    }
  }
}

template <typename U>
__device__ __forceinline__ double load_user(const void *p, int64_t i) {
  return double(static_cast<const U *>(p)[i]);
}

// one CTA per listed cell: user targets [n][3] / stiffness [n] -> SoA, targets kept in global coordinates (fp64)
template <typename T, typename U>
__global__ void __launch_bounds__(256)
set_collisions_kernel(const BucketView *__restrict__ views, const CellRef *__restrict__ refs, const CollisionDev *cols,
                      const void *__restrict__ targets, const void *__restrict__ stiffness) {
  const CellRef ref = refs[blockIdx.x];
  const BucketView bv = views[ref.bucket];
  const CollisionDev col = cols[ref.bucket];
  const int n = bv.n, n_pad = bv.n_pad;
  double *P = col.targets + size_t(ref.slot) * 3 * n_pad;
  T *W = static_cast<T *>(col.stiffness) + size_t(ref.slot) * n_pad;
  for (int i = threadIdx.x; i < 3 * n; i += blockDim.x)
    P[(i % 3) * n_pad + i / 3] = load_user<U>(targets, ref.user_offset + i);
  for (int i = threadIdx.x; i < n; i += blockDim.x) W[i] = T(load_user<U>(stiffness, ref.user_offset / 3 + i));
}

// g += k (x_n + d - p), one thread per (cell, vertex slot)
template <typename T>
__global__ void __launch_bounds__(256)
collision_grad_kernel(BucketView bv, CollisionDev col) {
  const T *x = static_cast<const T *>(bv.field[F_X]);
  const T *d = static_cast<const T *>(bv.field[F_D]);
  const T *xl = static_cast<const T *>(bv.field[F_XL]);      // null in fp64 contexts
  T *g = static_cast<T *>(bv.field[F_G]);
  const double *P = col.targets;
  const T *W = static_cast<const T *>(col.stiffness);
  const int n_pad = bv.n_pad;
  const size_t total = size_t(bv.cells) * n_pad;
  for (size_t i = blockIdx.x * size_t(blockDim.x) + threadIdx.x; i < total; i += size_t(gridDim.x) * blockDim.x) {
    const T w = W[i];
    if (w > T(0)) {
      const size_t cell = i / n_pad, base = cell * 3 * size_t(n_pad) + i % n_pad;
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        const size_t o = base + size_t(k) * n_pad;
        // the target in the cell's CURRENT local frame (fp64 difference of two global coordinates)
        const double local = (double(x[o]) + (xl ? double(xl[o]) : 0.0) + double(d[o])) - (P[o] - bv.origin[cell * 3 + k]);
        g[o] += w * T(local);
      }
    }
  }
}

// out[index of cell] += sum_i 1/2 k_i |x_i + d_i - p_i|^2, one warp per cell, fp64 accumulation
template <typename T>
__global__ void __launch_bounds__(128)
collision_energy_kernel(BucketView bv, CollisionDev col, const int64_t *__restrict__ cell_id, double *__restrict__ out,
                        const int *__restrict__ skip) {
  const int lane = threadIdx.x & 31;
  const int64_t warp0 = (int64_t(blockIdx.x) * blockDim.x + threadIdx.x) >> 5;
  const int64_t n_warps = (int64_t(gridDim.x) * blockDim.x) >> 5;
  const int n = bv.n, n_pad = bv.n_pad;
  if (skip && skip[bv.cells] == 0) return;              // line search: skip[cells] = cells still searching
  for (int64_t cell = warp0; cell < bv.cells; cell += n_warps) {
    if (skip && skip[cell]) continue;
    const size_t base = size_t(cell) * 3 * n_pad;
    const T *x = static_cast<const T *>(bv.field[F_X]) + base, *d = static_cast<const T *>(bv.field[F_D]) + base;
    const T *xl = bv.field[F_XL] ? static_cast<const T *>(bv.field[F_XL]) + base : nullptr;
    const double *P = col.targets + base;
    const double *origin = bv.origin + size_t(cell) * 3;
    const T *W = static_cast<const T *>(col.stiffness) + size_t(cell) * n_pad;
    double e = 0.0;
    for (int i = lane; i < n; i += 32) {
      const double w = double(W[i]);
      if (w > 0.0) {
        double r2 = 0.0;
        for (int k = 0; k < 3; ++k) {
          const double r = (double(x[k * n_pad + i]) + (xl ? double(xl[k * n_pad + i]) : 0.0) + double(d[k * n_pad + i])) -
                           (P[k * n_pad + i] - origin[k]);
          r2 += r * r;
        }
        e += 0.5 * w * r2;
      }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
    if (lane == 0) out[cell_id ? cell_id[cell] : cell] += e;
  }
}

}  // namespace

int launch_set_collisions(const BucketView *views_dev, const CollisionDev *cols_dev, const PackArgs &a, int precision,
                          cudaStream_t s) {
  if (a.n_refs == 0) return 0;
  const unsigned grid = unsigned(a.n_refs);
  if (precision == NPFEM_F32) {
    if (a.io_dtype == NPFEM_F32) set_collisions_kernel<float, float><<<grid, 256, 0, s>>>(views_dev, a.refs, cols_dev, a.src_a, a.src_b);
    else set_collisions_kernel<float, double><<<grid, 256, 0, s>>>(views_dev, a.refs, cols_dev, a.src_a, a.src_b);
  } else {
    if (a.io_dtype == NPFEM_F32) set_collisions_kernel<double, float><<<grid, 256, 0, s>>>(views_dev, a.refs, cols_dev, a.src_a, a.src_b);
    else set_collisions_kernel<double, double><<<grid, 256, 0, s>>>(views_dev, a.refs, cols_dev, a.src_a, a.src_b);
  }
  return 1;
}

int launch_collision_grad(const BucketView &bv, const CollisionDev &col, int precision, cudaStream_t s) {
  if (bv.cells == 0) return 0;
  const size_t total = size_t(bv.cells) * bv.n_pad;
  const unsigned grid = unsigned((total + 255) / 256 < 148 * 16 ? (total + 255) / 256 : 148 * 16);
  if (precision == NPFEM_F32) collision_grad_kernel<float><<<grid, 256, 0, s>>>(bv, col);
  else collision_grad_kernel<double><<<grid, 256, 0, s>>>(bv, col);
  return 1;
}

int launch_collision_energy(const BucketView &bv, const CollisionDev &col, const int64_t *cell_id_dev, double *out,
                            const int *skip_dev, int precision, cudaStream_t s) {
  if (bv.cells == 0) return 0;
  const int64_t ctas = (bv.cells + 3) / 4;
  const unsigned grid = unsigned(ctas < 148 * 16 ? ctas : 148 * 16);
  if (precision == NPFEM_F32) collision_energy_kernel<float><<<grid, 128, 0, s>>>(bv, col, cell_id_dev, out, skip_dev);
  else collision_energy_kernel<double><<<grid, 128, 0, s>>>(bv, col, cell_id_dev, out, skip_dev);
  return 1;
}

int launch_median_filter(const BucketView *views_dev, const CellRef *refs_dev, int64_t n_refs, int bucket,
                         const TypeDev &td, int precision, cudaStream_t s) {
  if (n_refs == 0) return 0;
  const size_t es = precision == NPFEM_F32 ? 4 : 8;
  const size_t smem = size_t(3) * td.n * es;
  if (smem > 200 * 1024 || td.valence_max > 32) return -1;
  if (precision == NPFEM_F32) {
    if (smem > 48 * 1024 &&   // off the hot path (once per set_forces): set every time, the attribute is per device
        cudaFuncSetAttribute(median_filter_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024) != cudaSuccess)
      return -1;
    median_filter_kernel<float><<<unsigned(n_refs), 256, smem, s>>>(views_dev, refs_dev, bucket, td.vtx_nbr, td.valence_max);
  } else {
    if (smem > 48 * 1024 &&
        cudaFuncSetAttribute(median_filter_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024) != cudaSuccess)
      return -1;
    median_filter_kernel<double><<<unsigned(n_refs), 256, smem, s>>>(views_dev, refs_dev, bucket, td.vtx_nbr, td.valence_max);
  }
  return 1;
}

}  // namespace npfem
