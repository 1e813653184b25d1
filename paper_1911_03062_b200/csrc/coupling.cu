// The solver's inputs from the fluid coupling that live on the solid side:
//   * median filter of F_ext over the one-ring of every vertex (reading R18: per vertex and
//     Cartesian component, the median over the vertex and its one-ring neighbours; an even count
//     averages the two central values), applied by npfem_set_forces when
//     NPFEM_OPT_FORCE_MEDIAN_FILTER is on;
//   * the vertex-velocity cap (reading R17) lives in the step epilogue (prologue.cu).
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

}  // namespace

int launch_median_filter(const BucketView *views_dev, const CellRef *refs_dev, int64_t n_refs, int bucket,
                         const TypeDev &td, int precision, cudaStream_t s) {
  if (n_refs == 0) return 0;
  const size_t es = precision == NPFEM_F32 ? 4 : 8;
  const size_t smem = size_t(3) * td.n * es;
  if (smem > 200 * 1024 || td.valence_max > 32) return -1;
  if (precision == NPFEM_F32) {
    if (smem > 48 * 1024 &&
        cudaFuncSetAttribute(median_filter_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem)) != cudaSuccess)
      return -1;
    median_filter_kernel<float><<<unsigned(n_refs), 256, smem, s>>>(views_dev, refs_dev, bucket, td.vtx_nbr, td.valence_max);
  } else {
    if (smem > 48 * 1024 &&
        cudaFuncSetAttribute(median_filter_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem)) != cudaSuccess)
      return -1;
    median_filter_kernel<double><<<unsigned(n_refs), 256, smem, s>>>(views_dev, refs_dev, bucket, td.vtx_nbr, td.valence_max);
  }
  return 1;
}

}  // namespace npfem
