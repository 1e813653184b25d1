// Dense fp64 inverse of the constant Hessian approximation H~ of one cell type, on the device.
//
// Eq. (4) (reading R1) needs H~^-1 applied every iteration; H~ is constant per
// cell TYPE, SPD and well conditioned (cond ~ 7-35 at h = 0.1 us), so it is inverted ONCE at
// creation by the Newton-Schulz iteration X <- X (2 I - H X), X0 = I / ||H||_inf, which is
// nothing but fp64 GEMMs (quadratic convergence; ~log2(cond)+6 iterations).  The final residual
// ||I - H X||_F is returned so that npfem_create can refuse a non-SPD / ill-conditioned system.
#include <cmath>
#include <cstdio>

#include "internal.h"

namespace npfem {
namespace {

constexpr int BM = 64, BN = 64, BK = 16;

// C = alpha * A * B + beta * D   (all n x n, row-major, leading dimension n)
__global__ void __launch_bounds__(256)
dgemm_nn_kernel(const double *__restrict__ A, const double *__restrict__ B, const double *__restrict__ D,
                double *__restrict__ C, int n, double alpha, double beta) {
  __shared__ double As[BK][BM + 1];
  __shared__ double Bs[BK][BN];
  const int tx = threadIdx.x % 16, ty = threadIdx.x / 16;
  const int row0 = blockIdx.y * BM, col0 = blockIdx.x * BN;
  double acc[4][4] = {};
  for (int k0 = 0; k0 < n; k0 += BK) {
    for (int i = threadIdx.x; i < BM * BK; i += 256) {
      const int r = i / BK, k = i % BK;
      As[k][r] = (row0 + r < n && k0 + k < n) ? A[size_t(row0 + r) * n + k0 + k] : 0.0;
    }
    for (int i = threadIdx.x; i < BK * BN; i += 256) {
      const int k = i / BN, c = i % BN;
      Bs[k][c] = (k0 + k < n && col0 + c < n) ? B[size_t(k0 + k) * n + col0 + c] : 0.0;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < BK; ++k) {
      double a[4], b[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) a[i] = As[k][ty + 16 * i];
#pragma unroll
      for (int j = 0; j < 4; ++j) b[j] = Bs[k][tx + 16 * j];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fma(a[i], b[j], acc[i][j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int r = row0 + ty + 16 * i, c = col0 + tx + 16 * j;
      if (r < n && c < n) {
        double v = alpha * acc[i][j];
        if (beta != 0.0) v += beta * D[size_t(r) * n + c];
        C[size_t(r) * n + c] = v;
      }
    }
}

__global__ void init_scaled_identity_kernel(double *X, int n, double s) {
  const size_t i = blockIdx.x * size_t(blockDim.x) + threadIdx.x;
  if (i < size_t(n) * n) X[i] = (i / n == i % n) ? s : 0.0;
}

// out[0] += sum (delta_ij - P_ij)^2
__global__ void identity_residual_kernel(const double *__restrict__ P, int n, double *out) {
  double acc = 0.0;
  for (size_t i = blockIdx.x * size_t(blockDim.x) + threadIdx.x; i < size_t(n) * n;
       i += size_t(gridDim.x) * blockDim.x) {
    const double r = ((i / n == i % n) ? 1.0 : 0.0) - P[i];
    acc += r * r;
  }
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if ((threadIdx.x & 31) == 0) atomicAdd(out, acc);
}

__global__ void symmetrise_kernel(const double *__restrict__ X, double *__restrict__ Y, int n) {
  const size_t i = blockIdx.x * size_t(blockDim.x) + threadIdx.x;
  if (i < size_t(n) * n) {
    const size_t r = i / n, c = i % n;
    Y[i] = 0.5 * (X[i] + X[c * n + r]);
  }
}

template <typename T>
__global__ void convert_pad_kernel(const double *__restrict__ X, int n, T *__restrict__ out, int n_pad) {
  const size_t i = blockIdx.x * size_t(blockDim.x) + threadIdx.x;
  if (i < size_t(n_pad) * n_pad) {
    const size_t r = i / n_pad, c = i % n_pad;
    out[i] = (r < size_t(n) && c < size_t(n)) ? T(X[r * n + c]) : T(0);
  }
}

}  // namespace

// out[n_pad][n_pad] (compute type) = X[n][n] (fp64), zero padded
__global__ void round_tf32_kernel(const float *__restrict__ in, float *__restrict__ out, size_t count) {
  for (size_t i = blockIdx.x * size_t(blockDim.x) + threadIdx.x; i < count; i += size_t(gridDim.x) * blockDim.x)
    out[i] = tf32_rn(in[i]);
}

int launch_round_tf32(const float *in, float *out, size_t count, cudaStream_t s) {
  if (count == 0) return 0;
  const unsigned grid = unsigned((count + 255) / 256 < 148 * 8 ? (count + 255) / 256 : 148 * 8);
  round_tf32_kernel<<<grid, 256, 0, s>>>(in, out, count);
  return 1;
}

int launch_convert_pad(const double *X, int n, void *out, int n_pad, int precision, cudaStream_t s) {
  const int eb = 256, eg = int((size_t(n_pad) * n_pad + eb - 1) / eb);
  if (precision == NPFEM_F32)
    convert_pad_kernel<float><<<eg, eb, 0, s>>>(X, n, static_cast<float *>(out), n_pad);
  else
    convert_pad_kernel<double><<<eg, eb, 0, s>>>(X, n, static_cast<double *>(out), n_pad);
  return 1;
}

// H_dev, Hinv_dev: device [n][n] fp64; tmp: invert_spd_tmp_doubles(n) doubles of device scratch.
// Synchronises the stream (setup path, called once per type).
size_t invert_spd_tmp_doubles(int n) { return size_t(3) * n * n + 32; }

int launch_invert_spd(const double *H_dev, double *Hinv_dev, int n, double *tmp, cudaStream_t stream,
                      double *residual_out, std::string &err) {
  int launches = 0;
  const size_t bytes = size_t(n) * n * sizeof(double);
  double *X = nullptr, *P = nullptr, *Y = nullptr, *res_dev = nullptr;
  std::vector<double> Hh(size_t(n) * n);
  if (cudaMemcpyAsync(Hh.data(), H_dev, bytes, cudaMemcpyDeviceToHost, stream) != cudaSuccess ||
      cudaStreamSynchronize(stream) != cudaSuccess) {
    err = "inverse: cannot read H~ back";
    return -1;
  }
  double norm_inf = 0.0;
  for (int r = 0; r < n; ++r) {
    double s = 0.0;
    for (int c = 0; c < n; ++c) s += std::fabs(Hh[size_t(r) * n + c]);
    norm_inf = s > norm_inf ? s : norm_inf;
    if (!(Hh[size_t(r) * n + r] > 0.0)) {
      err = "H~ has a non-positive diagonal entry: not SPD";
      return -1;
    }
  }
  // Newton-Schulz temporaries from the caller's scratch (workspace): no allocation here
  X = tmp;
  P = X + size_t(n) * n;
  Y = P + size_t(n) * n;
  res_dev = Y + size_t(n) * n;
  const dim3 grid((n + BN - 1) / BN, (n + BM - 1) / BM);
  const int eb = 256, eg = int((size_t(n) * n + eb - 1) / eb);
  init_scaled_identity_kernel<<<eg, eb, 0, stream>>>(X, n, 1.0 / norm_inf);
  ++launches;
  double res = 1e300, prev = 1e300;
  const double target = 1e-13 * std::sqrt(double(n));
  bool ok = false;
  for (int it = 0; it < 200; ++it) {
    dgemm_nn_kernel<<<grid, 256, 0, stream>>>(H_dev, X, nullptr, P, n, 1.0, 0.0);      // P = H X
    cudaMemsetAsync(res_dev, 0, sizeof(double), stream);
    identity_residual_kernel<<<296, 256, 0, stream>>>(P, n, res_dev);
    launches += 2;
    cudaMemcpyAsync(&res, res_dev, sizeof(double), cudaMemcpyDeviceToHost, stream);
    if (cudaStreamSynchronize(stream) != cudaSuccess) break;
    res = std::sqrt(res);
    if (!(res == res)) break;   // NaN
    if (res < target || (res < 1e-9 && res > 0.5 * prev)) {   // converged, or stagnated at round-off
      ok = true;
      break;
    }
    prev = res;
    dgemm_nn_kernel<<<grid, 256, 0, stream>>>(X, P, X, Y, n, -1.0, 2.0);               // Y = 2X - X (H X)
    ++launches;
    double *t = X; X = Y; Y = t;
  }
  if (ok) {
    symmetrise_kernel<<<eg, eb, 0, stream>>>(X, Hinv_dev, n);
    ++launches;
  }
  const cudaError_t e = cudaStreamSynchronize(stream);
  if (residual_out) *residual_out = res;
  if (e != cudaSuccess) {
    err = std::string("inverse: CUDA failure: ") + cudaGetErrorString(e);
    return -1;
  }
  if (!ok) {
    char buf[160];
    snprintf(buf, sizeof buf, "Newton-Schulz inverse of H~ did not converge (||I - H X||_F = %.3e): H~ not SPD or too ill-conditioned", res);
    err = buf;
    return -3;
  }
  return launches;
}

}  // namespace npfem
