// Measurement aid, not on the solver's path: a dependent-chain-free FFMA / DFMA loop whose launch bench.py --peaks
// times with CUDA events to MEASURE the plain-ALU roofs of the box the numbers were taken on (SURVEY.md 8(d):
// "measure an FFMA peak on the box"), instead of quoting 148 SMs x 128 lanes x 2 x the nominal clock.
#include "internal.h"

namespace npfem {
namespace {

// 16 independent accumulator chains per thread: enough ILP to keep one FMA per lane and cycle in flight
template <typename T>
__global__ void __launch_bounds__(256) fma_peak_kernel(T *__restrict__ sink, int iterations, T a, T b) {
  T acc[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) acc[i] = T(threadIdx.x + i);
  for (int it = 0; it < iterations; ++it) {
#pragma unroll
    for (int i = 0; i < 16; ++i) acc[i] = fma(acc[i], a, b);
  }
  T s = T(0);
#pragma unroll
  for (int i = 0; i < 16; ++i) s += acc[i];
  if (s == T(-1.2345)) sink[0] = s;                     // never true: keeps the loop alive
}

}  // namespace
}  // namespace npfem

extern "C" {

// Enqueue the probe on `cuda_stream`: grid_ctas CTAs of 256 threads, each thread 16 * iterations FMAs of the given
// precision (NPFEM_F32 / NPFEM_F64).  flops_out (HOST, may be NULL) receives 2 * 16 * iterations * 256 * grid_ctas.
// sink_dev: DEVICE scalar of that precision (never written in practice).  Returns NPFEM_OK or NPFEM_EINVAL / NPFEM_ECUDA.
int npfem_probe_fma_peak(void *cuda_stream, int32_t precision, int32_t grid_ctas, int32_t iterations, void *sink_dev,
                         double *flops_out) {
  if (grid_ctas < 1 || iterations < 1 || !sink_dev || (precision != NPFEM_F32 && precision != NPFEM_F64)) return NPFEM_EINVAL;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  if (precision == NPFEM_F32)
    npfem::fma_peak_kernel<float><<<unsigned(grid_ctas), 256, 0, s>>>(static_cast<float *>(sink_dev), iterations, 0.999f, 1e-3f);
  else
    npfem::fma_peak_kernel<double><<<unsigned(grid_ctas), 256, 0, s>>>(static_cast<double *>(sink_dev), iterations, 0.999, 1e-3);
  if (flops_out) *flops_out = 2.0 * 16.0 * double(iterations) * 256.0 * double(grid_ctas);
  return cudaGetLastError() == cudaSuccess ? NPFEM_OK : NPFEM_ECUDA;
}

}  // extern "C"
