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

// 16-byte accesses over the PADDED rows (n_pad is a multiple of 16, padding columns are zero in every field)
template <typename T> struct Vec16;
template <> struct Vec16<float> { typedef float4 type; };
template <> struct Vec16<double> { typedef double2 type; };

template <typename T>
__global__ void __launch_bounds__(128)
ls_init_kernel(BucketView bv, LineSearchDev ls, double grad_tol) {
  typedef typename Vec16<T>::type V;
  constexpr int W = int(sizeof(V) / sizeof(T));
  const int lane = threadIdx.x & 31;
  const int64_t warp0 = (int64_t(blockIdx.x) * blockDim.x + threadIdx.x) >> 5;
  const int64_t n_warps = (int64_t(gridDim.x) * blockDim.x) >> 5;
  const int nv = 3 * bv.n_pad / W;               // vectors per cell
  for (int64_t cell = warp0; cell < bv.cells; cell += n_warps) {
    const size_t base = size_t(cell) * 3 * bv.n_pad;
    V *g = reinterpret_cast<V *>(static_cast<T *>(bv.field[F_G]) + base);
    V *d = reinterpret_cast<V *>(static_cast<T *>(bv.field[F_D]) + base);
    const V *d_old = reinterpret_cast<const V *>(static_cast<const T *>(ls.d_old) + base);
    const V *b = reinterpret_cast<const V *>(static_cast<const T *>(bv.field[F_B]) + base);
    const float4 *g_lo = ls.g_lo ? reinterpret_cast<const float4 *>(ls.g_lo + base) : nullptr;   // 3xTF32 mode: gradient = g + g_lo
    double slope = 0.0, gg = 0.0, bb = 0.0;
    for (int i = lane; i < nv; i += 32) {
      V gv = g[i];
      const V dv = d[i], ov = d_old[i], bv4 = b[i];
      T *ge = reinterpret_cast<T *>(&gv);
      const T *de = reinterpret_cast<const T *>(&dv), *oe = reinterpret_cast<const T *>(&ov), *be = reinterpret_cast<const T *>(&bv4);
      float lo[4] = {0.f, 0.f, 0.f, 0.f};
      if (sizeof(T) == 4 && g_lo) *reinterpret_cast<float4 *>(lo) = g_lo[i];
#pragma unroll
      for (int e = 0; e < W; ++e) {
        const T p = de[e] - oe[e];                // the search direction, rounded once to the compute type
        const double gi = double(ge[e]) + double(lo[e]), bi = double(be[e]);
        slope += gi * double(p);
        gg += gi * gi;
        bb += bi * bi;
        ge[e] = p;                                // the gradient is not needed any more: keep p in its place
      }
      g[i] = gv;
    }
    slope = warp_sum(slope);
    gg = warp_sum(gg);
    bb = warp_sum(bb);
    const bool frozen = sqrt(gg) <= grad_tol * sqrt(bb);
    if (frozen)
      for (int i = lane; i < nv; i += 32) d[i] = d_old[i];
    if (lane == 0) {
      ls.slope[cell] = slope;
      ls.alpha[cell] = frozen ? 0.0 : 1.0;
      ls.done[cell] = frozen ? 1 : 0;
      if (!frozen) atomicAdd(ls.done + bv.cells, 1);     // cells still searching (zeroed by launch_ls_init)
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
  if (*static_cast<volatile const int *>(ls.done + bv.cells) == 0) return;   // every cell has settled: nothing to do
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
        atomicSub(ls.done + bv.cells, 1);
      }
      continue;
    }
    const double half = 0.5 * alpha;
    const size_t base = size_t(cell) * 3 * n_pad;
    const T *p = static_cast<const T *>(bv.field[F_G]) + base;
    T *d = static_cast<T *>(bv.field[F_D]) + base;
    const T *d_old = static_cast<const T *>(ls.d_old) + base;
    for (int k = 0; k < 3; ++k)
      for (int i = lane; i < n; i += 32) {
        const int o = k * n_pad + i;
        d[o] = d_old[o] + T(half) * p[o];       // alpha is a power of two: the product is exact
      }
    if (lane == 0) ls.alpha[cell] = half;
  }
}

// The fast local-step kernels store the REDUCED gradient r = (1 - gamma) m^ d - b + grad E; the
// line search needs the full one (slope, gradient norm; the global step then runs with d_scale = 1):
//   grad g = r + gamma m^ d + (beta/h) L z,   z = k_mem d + k_b A^-1 L d   (L = cotangent stencil)
// One CTA per cell, d and z in shared memory; same arithmetic order as the generic local step's stencil.
struct DampingParams {
  int n, n_pad, valence_max, g_tf32;
  const int *vtx_nbr;
  const float *vtx_w, *vtx_mass, *vtx_inv_area;
  float k_mem, k_b, beta_over_h, gamma_inertia;   // gamma (1 + h alpha) / h^2
  const float *d;
  float *g;
  float *g_lo;                                     // != nullptr: g <- tf32(grad), g_lo <- tf32(grad - g) (3xTF32 operands)
  int64_t cells;
};

__global__ void __launch_bounds__(256)
damping_grad_kernel(const DampingParams p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int n = p.n, n_pad = p.n_pad;
  float *sd = reinterpret_cast<float *>(smem_raw);   // [3][n]
  float *sz = sd + 3 * n;                             // [3][n]
  for (int64_t cell = blockIdx.x; cell < p.cells; cell += gridDim.x) {
    const size_t base = size_t(cell) * 3 * n_pad;
    for (int k = 0; k < 3; ++k)
      for (int i = threadIdx.x; i < n; i += blockDim.x) sd[k * n + i] = p.d[base + k * n_pad + i];
    __syncthreads();
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
      const float w0 = p.vtx_w[i];
      float u[3] = {w0 * sd[i], w0 * sd[n + i], w0 * sd[2 * n + i]};
      for (int q = 0; q < p.valence_max; ++q) {
        const int j = p.vtx_nbr[q * n + i];
        const float w = p.vtx_w[(q + 1) * n + i];
        u[0] += w * sd[j];
        u[1] += w * sd[n + j];
        u[2] += w * sd[2 * n + j];
      }
      const float s = p.k_b * p.vtx_inv_area[i];
      for (int k = 0; k < 3; ++k) sz[k * n + i] = p.k_mem * sd[k * n + i] + s * u[k];
    }
    __syncthreads();
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
      const float w0 = p.vtx_w[i];
      float lz[3] = {w0 * sz[i], w0 * sz[n + i], w0 * sz[2 * n + i]};
      for (int q = 0; q < p.valence_max; ++q) {
        const int j = p.vtx_nbr[q * n + i];
        const float w = p.vtx_w[(q + 1) * n + i];
        for (int k = 0; k < 3; ++k) lz[k] += w * sz[k * n + j];
      }
      const float mi = p.gamma_inertia * p.vtx_mass[i];
      for (int k = 0; k < 3; ++k) {
        const float gk = p.g[base + k * n_pad + i] + mi * sd[k * n + i] + p.beta_over_h * lz[k];
        if (p.g_lo) {
          const float hi = tf32_rn(gk);
          p.g[base + k * n_pad + i] = hi;
          p.g_lo[base + k * n_pad + i] = tf32_rn(gk - hi);
        } else {
          p.g[base + k * n_pad + i] = p.g_tf32 ? tf32_rn(gk) : gk;
        }
      }
    }
    __syncthreads();
  }
}

// The same for cells of at most 768 vertices (RBC-642, PLT-162): persistent CTAs, the one-ring tables of the thread's
// <= 3 vertices (neighbour ids packed in pairs, weights, inverse area, mass) live in REGISTERS for the whole launch
// instead of coming from L1 / L2 twice per cell, and the cell's g is requested together with its d at the top of the
// cell, so its latency runs under the two stencil passes (ncu on the plain kernel: long-scoreboard 15 per issue).
// Same arithmetic in the same order: bit-identical to damping_grad_kernel.
template <int MAXQ>
__global__ void __launch_bounds__(256, 2)
damping_grad_reg_kernel(const DampingParams p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int VPT = 3;
  const int n = p.n, n_pad = p.n_pad;
  float *sd = reinterpret_cast<float *>(smem_raw);   // [3][n]
  float *sz = sd + 3 * n;                             // [3][n]
  uint32_t nb[VPT][MAXQ / 2];
  float w[VPT][MAXQ + 1], ks[VPT], mi[VPT];
#pragma unroll
  for (int v = 0; v < VPT; ++v) {
    const int i = threadIdx.x + 256 * v;
    const bool a = i < n;
    w[v][0] = a ? p.vtx_w[i] : 0.f;
#pragma unroll
    for (int q = 0; q < MAXQ; q += 2) {
      const int j0 = a && q < p.valence_max ? p.vtx_nbr[q * n + i] : 0;
      const int j1 = a && q + 1 < p.valence_max ? p.vtx_nbr[(q + 1) * n + i] : 0;
      nb[v][q / 2] = uint32_t(j0) | (uint32_t(j1) << 16);
      w[v][q + 1] = a && q < p.valence_max ? p.vtx_w[(q + 1) * n + i] : 0.f;
      w[v][q + 2] = a && q + 1 < p.valence_max ? p.vtx_w[(q + 2) * n + i] : 0.f;
    }
    ks[v] = a ? p.k_b * p.vtx_inv_area[i] : 0.f;
    mi[v] = a ? p.gamma_inertia * p.vtx_mass[i] : 0.f;
  }
  for (int64_t cell = blockIdx.x; cell < p.cells; cell += gridDim.x) {
    const size_t base = size_t(cell) * 3 * n_pad;
    float gk[VPT][3];
#pragma unroll
    for (int v = 0; v < VPT; ++v) {
      const int i = threadIdx.x + 256 * v;
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        if (i < n) sd[k * n + i] = p.d[base + k * n_pad + i];
        gk[v][k] = i < n ? p.g[base + k * n_pad + i] : 0.f;
      }
    }
    __syncthreads();
#pragma unroll
    for (int v = 0; v < VPT; ++v) {
      const int i = threadIdx.x + 256 * v;
      if (i < n) {
        float u[3] = {w[v][0] * sd[i], w[v][0] * sd[n + i], w[v][0] * sd[2 * n + i]};
#pragma unroll
        for (int q = 0; q < MAXQ; ++q)
          if (q < p.valence_max) {
            const int j = int((q & 1) ? nb[v][q / 2] >> 16 : nb[v][q / 2] & 0xffffu);
            const float wq = w[v][q + 1];
            u[0] += wq * sd[j];
            u[1] += wq * sd[n + j];
            u[2] += wq * sd[2 * n + j];
          }
#pragma unroll
        for (int k = 0; k < 3; ++k) sz[k * n + i] = p.k_mem * sd[k * n + i] + ks[v] * u[k];
      }
    }
    __syncthreads();
#pragma unroll
    for (int v = 0; v < VPT; ++v) {
      const int i = threadIdx.x + 256 * v;
      if (i < n) {
        float lz[3] = {w[v][0] * sz[i], w[v][0] * sz[n + i], w[v][0] * sz[2 * n + i]};
#pragma unroll
        for (int q = 0; q < MAXQ; ++q)
          if (q < p.valence_max) {
            const int j = int((q & 1) ? nb[v][q / 2] >> 16 : nb[v][q / 2] & 0xffffu);
            const float wq = w[v][q + 1];
#pragma unroll
            for (int k = 0; k < 3; ++k) lz[k] += wq * sz[k * n + j];
          }
#pragma unroll
        for (int k = 0; k < 3; ++k) {
          const float g = gk[v][k] + mi[v] * sd[k * n + i] + p.beta_over_h * lz[k];
          if (p.g_lo) {
            const float hi = tf32_rn(g);
            p.g[base + k * n_pad + i] = hi;
            p.g_lo[base + k * n_pad + i] = tf32_rn(g - hi);
          } else {
            p.g[base + k * n_pad + i] = p.g_tf32 ? tf32_rn(g) : g;
          }
        }
      }
    }
    __syncthreads();
  }
}

__global__ void __launch_bounds__(256) split_g_kernel(float *__restrict__ g, float *__restrict__ g_lo, size_t count) {
  for (size_t i = size_t(blockIdx.x) * blockDim.x + threadIdx.x; i < count; i += size_t(gridDim.x) * blockDim.x) {
    const float v = g[i], hi = tf32_rn(v);
    g[i] = hi;
    g_lo[i] = tf32_rn(v - hi);
  }
}
__global__ void __launch_bounds__(256) split_w_kernel(const float *__restrict__ w, const float *__restrict__ w_hi,
                                                     float *__restrict__ w_lo, size_t count) {
  for (size_t i = size_t(blockIdx.x) * blockDim.x + threadIdx.x; i < count; i += size_t(gridDim.x) * blockDim.x)
    w_lo[i] = tf32_rn(w[i] - w_hi[i]);
}

unsigned warp_grid(int64_t cells) {
  const int64_t ctas = (cells + 3) / 4;
  return unsigned(ctas < 148 * 16 ? ctas : 148 * 16);
}

}  // namespace

int launch_damping_grad(const TypeDev &td, const BucketView &bv, float *g_lo, int n_sm, cudaStream_t s) {
  if (bv.cells == 0) return 0;
  if (td.beta_over_h == 0.0)   // nothing to add: only the split, if asked for
    return g_lo ? launch_ls_split_g(static_cast<float *>(bv.field[F_G]), g_lo, size_t(bv.cells) * 3 * td.n_pad, s) : 0;
  DampingParams p;
  p.n = td.n; p.n_pad = td.n_pad; p.valence_max = td.valence_max; p.g_tf32 = bv.g_tf32;
  p.vtx_nbr = td.vtx_nbr;
  p.vtx_w = static_cast<const float *>(td.vtx_w);
  p.vtx_mass = static_cast<const float *>(td.vtx_mass);
  p.vtx_inv_area = static_cast<const float *>(td.vtx_inv_area);
  p.k_mem = float(td.k_mem); p.k_b = float(td.k_b); p.beta_over_h = float(td.beta_over_h);
  p.gamma_inertia = float(td.gamma * td.inertia_coef);
  p.d = static_cast<const float *>(bv.field[F_D]);
  p.g = static_cast<float *>(bv.field[F_G]);
  p.g_lo = g_lo;
  p.cells = bv.cells;
  const size_t smem = sizeof(float) * 6 * size_t(td.n);
  if (smem > 200 * 1024) return -1;
  if (!td.cache.damping_attr) cudaFuncSetAttribute(damping_grad_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
  td.cache.damping_attr = true;
  if (td.n <= 768 && td.valence_max <= 8) {   // tables in registers, persistent: 2 CTAs per SM (registers)
    const int64_t capr = int64_t(n_sm) * 2;
    damping_grad_reg_kernel<8><<<unsigned(bv.cells < capr ? bv.cells : capr), 256, smem, s>>>(p);
    return 1;
  }
  const int64_t cap = int64_t(n_sm) * 8 * 2;
  damping_grad_kernel<<<unsigned(bv.cells < cap ? bv.cells : cap), 256, smem, s>>>(p);
  return 1;
}

int launch_ls_split_g(float *g, float *g_lo, size_t count, cudaStream_t s) {
  if (count == 0) return 0;
  const size_t ctas = (count + 1023) / 1024;
  split_g_kernel<<<unsigned(ctas < 148 * 16 ? ctas : 148 * 16), 256, 0, s>>>(g, g_lo, count);
  return 1;
}

int launch_ls_split_w(const float *w, const float *w_hi, float *w_lo, size_t count, cudaStream_t s) {
  if (count == 0) return 0;
  const size_t ctas = (count + 1023) / 1024;
  split_w_kernel<<<unsigned(ctas < 148 * 16 ? ctas : 148 * 16), 256, 0, s>>>(w, w_hi, w_lo, count);
  return 1;
}

int launch_ls_init(const BucketView &bv, const LineSearchDev &ls, double grad_tol, int precision, cudaStream_t s) {
  if (bv.cells == 0) return 0;
  if (cudaMemsetAsync(ls.done + bv.cells, 0, sizeof(int), s) != cudaSuccess) return -2;
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
