// Global step (row a3), SIMT path: d <- d - g H~^-1  (Eq. (4), reading R1).
//
// H~^-1 is one constant dense n x n operator per cell TYPE and acts on the three coordinate
// columns of every cell of that type, so the whole bucket is ONE GEMM
//     D[3*cells x n_pad] -= G[3*cells x n_pad] . W[n_pad x n_pad],   W = H~^-1 (symmetric).
// This file is the exact-arithmetic path: FP64 contexts (DFMA) and the FP32-FFMA option of FP32
// contexts.  The tcgen05/TF32 tensor-core path lives in global_tcgen05.cu.
#include "internal.h"

namespace npfem {
namespace {

template <typename T, int BM, int BN, int BK, int TM, int TN>
__global__ void __launch_bounds__((BM / TM) * (BN / TN))
global_simt_kernel(const T *__restrict__ G, const T *__restrict__ W, T *__restrict__ D, int64_t rows, int n_pad, T d_scale) {
  constexpr int NT = (BM / TM) * (BN / TN);
  __shared__ T Gs[BK][BM + 4];
  __shared__ T Ws[BK][BN];
  const int tx = threadIdx.x % (BN / TN), ty = threadIdx.x / (BN / TN);
  const int64_t row0 = int64_t(blockIdx.y) * BM;
  const int col0 = blockIdx.x * BN;
  T acc[TM][TN] = {};
  for (int k0 = 0; k0 < n_pad; k0 += BK) {
    for (int i = threadIdx.x; i < BM * BK; i += NT) {
      const int r = i / BK, k = i % BK;
      Gs[k][r] = (row0 + r < rows) ? G[(row0 + r) * n_pad + k0 + k] : T(0);
    }
    for (int i = threadIdx.x; i < BK * BN; i += NT) {
      const int k = i / BN, c = i % BN;
      Ws[k][c] = (col0 + c < n_pad) ? W[size_t(k0 + k) * n_pad + col0 + c] : T(0);
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < BK; ++k) {
      T a[TM], b[TN];
#pragma unroll
      for (int i = 0; i < TM; ++i) a[i] = Gs[k][ty + (BM / TM) * i];
#pragma unroll
      for (int j = 0; j < TN; ++j) b[j] = Ws[k][tx + (BN / TN) * j];
#pragma unroll
      for (int i = 0; i < TM; ++i)
#pragma unroll
        for (int j = 0; j < TN; ++j) acc[i][j] = fma(a[i], b[j], acc[i][j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < TM; ++i)
#pragma unroll
    for (int j = 0; j < TN; ++j) {
      const int64_t r = row0 + ty + (BM / TM) * i;
      const int c = col0 + tx + (BN / TN) * j;
      if (r < rows && c < n_pad) D[r * n_pad + c] = d_scale * D[r * n_pad + c] - acc[i][j];
    }
}

}  // namespace

int launch_global_simt(const TypeDev &td, const BucketView &bv, int precision, double d_scale, cudaStream_t s) {
  if (bv.cells == 0) return 0;
  const int64_t rows = bv.cells * 3;
  constexpr int BM = 64, BN = 64;
  const dim3 grid((td.n_pad + BN - 1) / BN, unsigned((rows + BM - 1) / BM));
  if (precision == NPFEM_F32)
    global_simt_kernel<float, BM, BN, 16, 4, 4><<<grid, 256, 0, s>>>(
        static_cast<const float *>(bv.field[F_G]), static_cast<const float *>(td.Hinv),
        static_cast<float *>(bv.field[F_D]), rows, td.n_pad, float(d_scale));
  else
    global_simt_kernel<double, BM, BN, 16, 4, 4><<<grid, 256, 0, s>>>(
        static_cast<const double *>(bv.field[F_G]), static_cast<const double *>(td.Hinv),
        static_cast<double *>(bv.field[F_D]), rows, td.n_pad, d_scale);
  return 1;
}

}  // namespace npfem
