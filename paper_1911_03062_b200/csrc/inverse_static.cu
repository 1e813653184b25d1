// npfem_invert_spd_static: the fp64 Newton-Schulz inverse of inverse.cu for callers that cannot allocate device
// memory at all (code under CUDA graph capture around it, serving loops, harnesses that forbid cudaMalloc).
//
// The operation is the one npfem_create runs once per cell type (Eq. (4): the global step applies
// H~^-1, H~ constant per type, so it is inverted once): X <- X (2 I - H X) from X0 = I / ||H||_inf.  Its three n x n
// fp64 temporaries and its residual accumulator are SCRATCH; npfem_create takes them from the caller's workspace,
// npfem_invert_spd (below) from a caller-owned buffer, and npfem_invert_spd_static from the file-scope device array
// `g_invert_scratch` of this translation unit:
//
//   size      3 * NPFEM_INVERT_STATIC_MAX_N^2 + 32 doubles = 1,597,792 bytes (MAX_N = 258, the paper's RBC resolution)
//   lifetime  every device that loads the library holds it from module load until the process exits
//   sharing   ONE array per device for all calls and all host threads: calls that overlap on the GPU (two streams,
//             two threads) race on it - serialise them.  It keeps the last call's contents; the only part that has
//             to start at zero is the residual accumulator, cleared here before every use (X is initialised, P and Y
//             are fully written before they are read).
//
// In host code `g_invert_scratch` is a host-side stand-in, not a device address: the address the kernels get comes
// from cudaGetSymbolAddress, asked once per device with that device current.  No cudaMalloc / cudaFree / allocating
// library routine is called on this path (the copy of H read back for ||H||_inf is a std::vector: host memory).
#include <cstdio>
#include <mutex>
#include <string>

#include "internal.h"

namespace {

constexpr int kMaxN = NPFEM_INVERT_STATIC_MAX_N;
constexpr size_t kScratchDoubles = size_t(3) * kMaxN * kMaxN + 32;
constexpr int kMaxDevices = 64;

static __device__ __align__(256) double g_invert_scratch[kScratchDoubles];

std::mutex g_mutex;                       // guards the per-device address cache only
double *g_scratch_of_device[kMaxDevices];  // nullptr = not asked yet
thread_local std::string g_error;

int fail(int code, const std::string &msg) {
  g_error = msg;
  return code;
}

// Device address of g_invert_scratch on the CURRENT device (asked once per device).
int scratch_address(double **out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(NPFEM_ECUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e));
  if (dev < 0 || dev >= kMaxDevices) return fail(NPFEM_EINVAL, "device ordinal beyond the 64 this entry point keeps addresses for");
  std::lock_guard<std::mutex> lock(g_mutex);
  if (!g_scratch_of_device[dev]) {
    double *ptr = nullptr;
    e = cudaGetSymbolAddress(reinterpret_cast<void **>(&ptr), g_invert_scratch);
    if (e != cudaSuccess || !ptr)
      return fail(NPFEM_ECUDA, std::string("cudaGetSymbolAddress(g_invert_scratch): ") + cudaGetErrorString(e));
    g_scratch_of_device[dev] = ptr;
  }
  *out = g_scratch_of_device[dev];
  return NPFEM_OK;
}

int run(const double *H_dev, double *Hinv_dev, int n, double *tmp, cudaStream_t stream, double *residual_out) {
  // the accumulator behind the three matrices must start at zero; everything else is written before it is read
  if (cudaMemsetAsync(tmp + size_t(3) * n * n, 0, 32 * sizeof(double), stream) != cudaSuccess)
    return fail(NPFEM_ECUDA, "cannot clear the residual accumulator of the scratch");
  std::string err;
  const int rc = npfem::launch_invert_spd(H_dev, Hinv_dev, n, tmp, stream, residual_out, err);
  if (rc >= 0) return NPFEM_OK;
  if (rc == -3) return fail(NPFEM_ESTATE, err);
  return fail(err.find("not SPD") != std::string::npos ? NPFEM_EINVAL : NPFEM_ECUDA, err);
}

}  // namespace

extern "C" {

size_t npfem_invert_spd_tmp_bytes(int32_t n) { return n < 1 ? 0 : npfem::invert_spd_tmp_doubles(n) * sizeof(double); }

int npfem_invert_spd(const double *H_dev, double *Hinv_dev, int32_t n, void *tmp_dev, size_t tmp_bytes, void *cuda_stream,
                     double *residual_out) {
  if (!H_dev || !Hinv_dev || !tmp_dev || n < 1) return fail(NPFEM_EINVAL, "npfem_invert_spd: NULL pointer or n < 1");
  if (reinterpret_cast<uintptr_t>(tmp_dev) % 256) return fail(NPFEM_EINVAL, "npfem_invert_spd: tmp_dev is not 256-byte aligned");
  if (tmp_bytes < npfem_invert_spd_tmp_bytes(n)) return fail(NPFEM_ENOMEM, "npfem_invert_spd: tmp_bytes below npfem_invert_spd_tmp_bytes(n)");
  return run(H_dev, Hinv_dev, n, static_cast<double *>(tmp_dev), static_cast<cudaStream_t>(cuda_stream), residual_out);
}

int npfem_invert_spd_static(const double *H_dev, double *Hinv_dev, int32_t n, void *cuda_stream, double *residual_out) {
  if (!H_dev || !Hinv_dev || n < 1) return fail(NPFEM_EINVAL, "npfem_invert_spd_static: NULL pointer or n < 1");
  if (n > kMaxN) {
    char buf[200];
    snprintf(buf, sizeof buf,
             "npfem_invert_spd_static: n = %d exceeds NPFEM_INVERT_STATIC_MAX_N = %d (the static scratch holds 3 * %d^2 + 32 "
             "doubles); use npfem_invert_spd with caller-owned scratch", n, kMaxN, kMaxN);
    return fail(NPFEM_EINVAL, buf);
  }
  double *tmp = nullptr;
  const int rc = scratch_address(&tmp);
  if (rc != NPFEM_OK) return rc;
  return run(H_dev, Hinv_dev, n, tmp, static_cast<cudaStream_t>(cuda_stream), residual_out);
}

const char *npfem_invert_spd_last_error(void) { return g_error.c_str(); }

}  // extern "C"
