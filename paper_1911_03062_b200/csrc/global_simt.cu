// Global step (row a3), SIMT path: d <- d - g H~^-1  (Eq. (4), reading R1).
//
// H~^-1 is one constant dense n x n operator per cell TYPE and acts on the three coordinate
// columns of every cell of that type, so the whole bucket is ONE GEMM
//     D[3*cells x n_pad] -= G[3*cells x n_pad] . W[n_pad x n_pad],   W = H~^-1 (symmetric).
// This file is the exact-arithmetic path: FP64 contexts (FP64 tensor cores, DMMA) and the FP32-FFMA
// option of FP32 contexts.  The tcgen05/TF32 tensor-core path lives in global_tcgen05.cu.
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

// FP64 contexts: the same GEMM on the FP64 tensor-core path (mma.sync m8n8k4, DMMA).  Block tile 128 x 64,
// 8 warps of 32 x 32 (4 x 4 MMA tiles, 32 accumulators per lane), BK = 16.  Shared-memory row strides of
// 20 / 68 doubles make the 64-bit fragment loads of a half warp hit 16 distinct banks.
__device__ __forceinline__ void dmma(double (&c)[2], double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
               : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}

__global__ void __launch_bounds__(256)
global_dmma_kernel(const double *__restrict__ G, const double *__restrict__ W, double *__restrict__ D, int64_t rows,
                   int n_pad, double d_scale) {
  constexpr int BM = 128, BN = 64, BK = 16, AS = BK + 4, BS = BN + 4;
  __shared__ double As[BM * AS];
  __shared__ double Bs[BK * BS];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = warp >> 1, wn = warp & 1;                 // 4 x 2 warps
  const int64_t row0 = int64_t(blockIdx.y) * BM;
  const int col0 = blockIdx.x * BN;
  double acc[4][4][2];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
  const int ar = tid >> 1, ak = (tid & 1) * 8;             // A tile: thread loads 8 consecutive doubles of row ar
  const int bk = tid >> 4, bc = (tid & 15) * 4;            // B tile: thread loads 4 consecutive doubles of row bk
  // register-prefetched pipeline: the next K-slice is loaded from global memory while the current one is multiplied
  const bool ok = row0 + ar < rows, okb = col0 + bc < n_pad;   // n_pad is a multiple of 16: a group of 4 is in or out
  const double2 *src = reinterpret_cast<const double2 *>(G + (row0 + ar) * n_pad + ak);
  const double2 *srcb = reinterpret_cast<const double2 *>(W + size_t(bk) * n_pad + col0 + bc);
  const double2 zero2 = make_double2(0.0, 0.0);
  double2 ra[4], rb[2];
#pragma unroll
  for (int q = 0; q < 4; ++q) ra[q] = ok ? src[q] : zero2;
#pragma unroll
  for (int q = 0; q < 2; ++q) rb[q] = okb ? srcb[q] : zero2;
  for (int k0 = 0; k0 < n_pad; k0 += BK) {
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      As[ar * AS + ak + 2 * q] = ra[q].x;
      As[ar * AS + ak + 2 * q + 1] = ra[q].y;
    }
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      Bs[bk * BS + bc + 2 * q] = rb[q].x;
      Bs[bk * BS + bc + 2 * q + 1] = rb[q].y;
    }
    __syncthreads();
    if (k0 + BK < n_pad) {
      const double2 *na = src + (k0 + BK) / 2;
      const double2 *nb = srcb + size_t(k0 + BK) * n_pad / 2;
#pragma unroll
      for (int q = 0; q < 4; ++q) ra[q] = ok ? na[q] : zero2;
#pragma unroll
      for (int q = 0; q < 2; ++q) rb[q] = okb ? nb[q] : zero2;
    }
#pragma unroll
    for (int kk = 0; kk < BK; kk += 4) {
      double a[4], b[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) a[i] = As[(wm * 32 + i * 8 + (lane >> 2)) * AS + kk + (lane & 3)];
#pragma unroll
      for (int j = 0; j < 4; ++j) b[j] = Bs[(kk + (lane & 3)) * BS + wn * 32 + j * 8 + (lane >> 2)];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) dmma(acc[i][j], a[i], b[j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int64_t r = row0 + wm * 32 + i * 8 + (lane >> 2);
      const int c = col0 + wn * 32 + j * 8 + 2 * (lane & 3);
      if (r < rows && c < n_pad) {
        double2 *dst = reinterpret_cast<double2 *>(D + r * n_pad + c);
        double2 v = *dst;
        v.x = d_scale * v.x - acc[i][j][0];
        v.y = d_scale * v.y - acc[i][j][1];
        *dst = v;
      }
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
  else {
    const dim3 grid64((td.n_pad + 63) / 64, unsigned((rows + 127) / 128));
    global_dmma_kernel<<<grid64, 256, 0, s>>>(static_cast<const double *>(bv.field[F_G]), static_cast<const double *>(td.Hinv),
                                              static_cast<double *>(bv.field[F_D]), rows, td.n_pad, d_scale);
  }
  return 1;
}

}  // namespace npfem
