// Step prologue (row a1) and epilogue (row a4).
//
// Prologue, once per time step and cell (readings R3, R12):
//   1. position-based-dynamics damping of v_n (paper's ref. [6]):
//        v <- v + kappa (v_cm + omega x r - v),  r = x - x_cm,
//        omega = I^-1 sum r x (m v),  I = sum m (|r|^2 Id - r r^T)
//   2. b = M v/h + F_ext  (so that grad g = M~ d/h^2 - b + grad E),  d^0 = h v.
//   It also re-centres the cell-local coordinates when the mass centre has drifted.
// Epilogue (Eq. 1): x_{n+1} = x_n + d, v_{n+1} = d/h.
#include "internal.h"

namespace npfem {
namespace {

template <int N>
__device__ __forceinline__ void block_sum_n(double (&v)[N], double *red /* [8][N] */) {
#pragma unroll
  for (int k = 0; k < N; ++k)
    for (int o = 16; o > 0; o >>= 1) v[k] += __shfl_xor_sync(0xffffffffu, v[k], o);
  const int w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  __syncthreads();
  if ((threadIdx.x & 31) == 0)
#pragma unroll
    for (int k = 0; k < N; ++k) red[w * N + k] = v[k];
  __syncthreads();
#pragma unroll
  for (int k = 0; k < N; ++k) {
    double s = 0.0;
    for (int i = 0; i < nw; ++i) s += red[i * N + k];
    v[k] = s;
  }
}

template <typename T>
__global__ void __launch_bounds__(256)
prologue_kernel(BucketView bv, const T *__restrict__ mass, double kappa, double h) {
  __shared__ double red[8 * 9];
  const int n = bv.n, n_pad = bv.n_pad;
  for (int64_t cell = blockIdx.x; cell < bv.cells; cell += gridDim.x) {
    const size_t base = size_t(cell) * 3 * n_pad;
    T *x = static_cast<T *>(bv.field[F_X]) + base;
    T *v = static_cast<T *>(bv.field[F_V]) + base;
    const T *f = static_cast<const T *>(bv.field[F_F]) + base;
    T *b = static_cast<T *>(bv.field[F_B]) + base;
    T *d = static_cast<T *>(bv.field[F_D]) + base;
    T *xl = bv.field[F_XL] ? static_cast<T *>(bv.field[F_XL]) + base : nullptr;

    double s[7] = {};   // sum m, sum m x, sum m v
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
      const double m = double(mass[i]);
      s[0] += m;
      for (int k = 0; k < 3; ++k) {
        s[1 + k] += m * double(x[k * n_pad + i]);
        s[4 + k] += m * double(v[k * n_pad + i]);
      }
    }
    block_sum_n<7>(s, red);
    const double xc[3] = {s[1] / s[0], s[2] / s[0], s[3] / s[0]};
    const double vc[3] = {s[4] / s[0], s[5] / s[0], s[6] / s[0]};

    double om[3] = {0.0, 0.0, 0.0};
    if (kappa > 0.0) {
      double q[9] = {};   // angular momentum (3), inertia xx yy zz xy xz yz
      for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const double m = double(mass[i]);
        const double r0 = double(x[i]) - xc[0], r1 = double(x[n_pad + i]) - xc[1], r2 = double(x[2 * n_pad + i]) - xc[2];
        const double p0 = m * double(v[i]), p1 = m * double(v[n_pad + i]), p2 = m * double(v[2 * n_pad + i]);
        q[0] += r1 * p2 - r2 * p1;
        q[1] += r2 * p0 - r0 * p2;
        q[2] += r0 * p1 - r1 * p0;
        q[3] += m * (r1 * r1 + r2 * r2);
        q[4] += m * (r0 * r0 + r2 * r2);
        q[5] += m * (r0 * r0 + r1 * r1);
        q[6] -= m * r0 * r1;
        q[7] -= m * r0 * r2;
        q[8] -= m * r1 * r2;
      }
      block_sum_n<9>(q, red);
      // omega = I^-1 L, symmetric 3x3 inverse by the adjugate
      const double a = q[3], bb = q[4], c = q[5], dxy = q[6], dxz = q[7], dyz = q[8];
      const double A00 = bb * c - dyz * dyz, A01 = dxz * dyz - dxy * c, A02 = dxy * dyz - dxz * bb;
      const double A11 = a * c - dxz * dxz, A12 = dxy * dxz - a * dyz, A22 = a * bb - dxy * dxy;
      const double det = a * A00 + dxy * A01 + dxz * A02;
      om[0] = (A00 * q[0] + A01 * q[1] + A02 * q[2]) / det;
      om[1] = (A01 * q[0] + A11 * q[1] + A12 * q[2]) / det;
      om[2] = (A02 * q[0] + A12 * q[1] + A22 * q[2]) / det;
    }

    // re-centre the local frame when the mass centre drifted (exact binary shift, rare)
    double shift[3] = {0.0, 0.0, 0.0};
    const bool recentre = fabs(xc[0]) > 0.5 || fabs(xc[1]) > 0.5 || fabs(xc[2]) > 0.5;
    if (recentre) {
      for (int k = 0; k < 3; ++k) shift[k] = rint(xc[k] * 1024.0) / 1024.0;
      if (threadIdx.x < 3) bv.origin[size_t(cell) * 3 + threadIdx.x] += shift[threadIdx.x];
    }

    for (int i = threadIdx.x; i < n; i += blockDim.x) {
      const double m = double(mass[i]);
      double xi[3], vi[3];
      for (int k = 0; k < 3; ++k) {
        xi[k] = double(x[k * n_pad + i]);
        vi[k] = double(v[k * n_pad + i]);
      }
      if (kappa > 0.0) {
        const double r0 = xi[0] - xc[0], r1 = xi[1] - xc[1], r2 = xi[2] - xc[2];
        const double w[3] = {om[1] * r2 - om[2] * r1, om[2] * r0 - om[0] * r2, om[0] * r1 - om[1] * r0};
        for (int k = 0; k < 3; ++k) vi[k] += kappa * (vc[k] + w[k] - vi[k]);
      }
      for (int k = 0; k < 3; ++k) {
        if (recentre) {   // what the shifted coordinate loses when it is rounded to T goes to the low part
          const T hi = T(xi[k] - shift[k]);
          x[k * n_pad + i] = hi;
          if (xl) xl[k * n_pad + i] += T((xi[k] - shift[k]) - double(hi));
        }
        v[k * n_pad + i] = T(vi[k]);
        b[k * n_pad + i] = T(m * vi[k] / h + double(f[k * n_pad + i]));
        d[k * n_pad + i] = T(h * vi[k]);
      }
    }
    __syncthreads();
  }
}

// fp32 fast path: ONE WARP per cell, the lane's vertices (x, v) stay in registers between the moment
// pass and the update pass, so every field is read and written once.  All 16 moments (mass, m x,
// m v, sum x x (m v), sum m x x^T about the local origin) are accumulated in fp64 in a single pass
// and shifted to the mass centre by the parallel-axis relations; the update itself runs in fp32.
template <int VPT>
__global__ void __launch_bounds__(128)
prologue_warp_kernel(BucketView bv, const float *__restrict__ mass, float kappa, float h) {
  const int n = bv.n, n_pad = bv.n_pad, lane = threadIdx.x & 31;
  const int64_t warp0 = (int64_t(blockIdx.x) * blockDim.x + threadIdx.x) >> 5;
  const int64_t n_warps = (int64_t(gridDim.x) * blockDim.x) >> 5;
  float m[VPT];
#pragma unroll
  for (int q = 0; q < VPT; ++q) m[q] = lane + 32 * q < n ? mass[lane + 32 * q] : 0.f;
  const float inv_h = 1.f / h;
  for (int64_t cell = warp0; cell < bv.cells; cell += n_warps) {
    const size_t base = size_t(cell) * 3 * n_pad;
    float *xg = static_cast<float *>(bv.field[F_X]) + base;
    float *vg = static_cast<float *>(bv.field[F_V]) + base;
    const float *fg = static_cast<const float *>(bv.field[F_F]) + base;
    float *bg = static_cast<float *>(bv.field[F_B]) + base;
    float *dg = static_cast<float *>(bv.field[F_D]) + base;
    float x[VPT][3], v[VPT][3];
#pragma unroll
    for (int q = 0; q < VPT; ++q) {
      const int i = lane + 32 * q;
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        x[q][k] = i < n ? __ldcs(xg + k * n_pad + i) : 0.f;
        v[q][k] = i < n ? __ldcs(vg + k * n_pad + i) : 0.f;
      }
    }
    double s[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) s[k] = 0.0;
#pragma unroll
    for (int q = 0; q < VPT; ++q) {
      const double md = double(m[q]);
      const double x0 = double(x[q][0]), x1 = double(x[q][1]), x2 = double(x[q][2]);
      const double p0 = md * double(v[q][0]), p1 = md * double(v[q][1]), p2 = md * double(v[q][2]);
      s[0] += md;
      s[1] += md * x0; s[2] += md * x1; s[3] += md * x2;
      s[4] += p0; s[5] += p1; s[6] += p2;
      if (kappa > 0.f) {
        s[7] += x1 * p2 - x2 * p1; s[8] += x2 * p0 - x0 * p2; s[9] += x0 * p1 - x1 * p0;
        s[10] += md * x0 * x0; s[11] += md * x1 * x1; s[12] += md * x2 * x2;
        s[13] += md * x0 * x1; s[14] += md * x0 * x2; s[15] += md * x1 * x2;
      }
    }
    const int n_red = kappa > 0.f ? 16 : 7;
#pragma unroll
    for (int k = 0; k < 16; ++k)
      if (k < n_red)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s[k] += __shfl_xor_sync(0xffffffffu, s[k], o);
    const double M = s[0], inv_M = 1.0 / M;
    const double xc[3] = {s[1] * inv_M, s[2] * inv_M, s[3] * inv_M};
    const double vc[3] = {s[4] * inv_M, s[5] * inv_M, s[6] * inv_M};
    double om[3] = {0.0, 0.0, 0.0};
    if (kappa > 0.f) {
      // about the mass centre: L_c = L_0 - x_c x P,  S_c = S_0 - M x_c x_c^T
      const double L0 = s[7] - (xc[1] * s[6] - xc[2] * s[5]);
      const double L1 = s[8] - (xc[2] * s[4] - xc[0] * s[6]);
      const double L2 = s[9] - (xc[0] * s[5] - xc[1] * s[4]);
      const double Sxx = s[10] - M * xc[0] * xc[0], Syy = s[11] - M * xc[1] * xc[1], Szz = s[12] - M * xc[2] * xc[2];
      const double a = Syy + Szz, bb = Sxx + Szz, c = Sxx + Syy;
      const double dxy = -(s[13] - M * xc[0] * xc[1]), dxz = -(s[14] - M * xc[0] * xc[2]), dyz = -(s[15] - M * xc[1] * xc[2]);
      const double A00 = bb * c - dyz * dyz, A01 = dxz * dyz - dxy * c, A02 = dxy * dyz - dxz * bb;
      const double A11 = a * c - dxz * dxz, A12 = dxy * dxz - a * dyz, A22 = a * bb - dxy * dxy;
      const double inv_det = 1.0 / (a * A00 + dxy * A01 + dxz * A02);
      om[0] = (A00 * L0 + A01 * L1 + A02 * L2) * inv_det;
      om[1] = (A01 * L0 + A11 * L1 + A12 * L2) * inv_det;
      om[2] = (A02 * L0 + A12 * L1 + A22 * L2) * inv_det;
    }
    // re-centre the local frame when the mass centre drifted (exact binary shift, rare)
    float shift[3] = {0.f, 0.f, 0.f};
    const bool recentre = fabs(xc[0]) > 0.5 || fabs(xc[1]) > 0.5 || fabs(xc[2]) > 0.5;
    if (recentre) {
      double sh[3];
#pragma unroll
      for (int k = 0; k < 3; ++k) { sh[k] = rint(xc[k] * 1024.0) / 1024.0; shift[k] = float(sh[k]); }
      if (lane < 3) bv.origin[size_t(cell) * 3 + lane] += lane == 0 ? sh[0] : (lane == 1 ? sh[1] : sh[2]);
    }
    const float xcf[3] = {float(xc[0]), float(xc[1]), float(xc[2])}, vcf[3] = {float(vc[0]), float(vc[1]), float(vc[2])};
    const float omf[3] = {float(om[0]), float(om[1]), float(om[2])};
    // three separate loops so that the F loads are issued back to back (a store between two loads
    // would serialise them on a full DRAM latency each)
#pragma unroll
    for (int q = 0; q < VPT; ++q) {
      const int i = lane + 32 * q;
      if (kappa > 0.f) {
        const float r0 = x[q][0] - xcf[0], r1 = x[q][1] - xcf[1], r2 = x[q][2] - xcf[2];
        const float w[3] = {omf[1] * r2 - omf[2] * r1, omf[2] * r0 - omf[0] * r2, omf[0] * r1 - omf[1] * r0};
#pragma unroll
        for (int k = 0; k < 3; ++k) v[q][k] += kappa * (vcf[k] + w[k] - v[q][k]);
      }
      if (recentre && i < n) {   // rare; the rounding of the shifted coordinate goes to the low part (F_XL)
        float *xlg = static_cast<float *>(bv.field[F_XL]) + base;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
          const double xs = double(x[q][k]) - double(shift[k]);
          const float hi = float(xs);
          xg[k * n_pad + i] = hi;
          xlg[k * n_pad + i] += float(xs - double(hi));
        }
      }
    }
    float f[VPT][3];
#pragma unroll
    for (int q = 0; q < VPT; ++q) {
      const int i = lane + 32 * q;
#pragma unroll
      for (int k = 0; k < 3; ++k) f[q][k] = i < n ? __ldcs(fg + k * n_pad + i) : 0.f;
    }
#pragma unroll
    for (int q = 0; q < VPT; ++q) {
      const int i = lane + 32 * q;
      if (i < n) {
        const float mh = m[q] * inv_h;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
          vg[k * n_pad + i] = v[q][k];
          bg[k * n_pad + i] = fmaf(mh, v[q][k], f[q][k]);
          dg[k * n_pad + i] = h * v[q][k];
        }
      }
    }
  }
}

// x_{n+1} = x_n + d, v_{n+1} = d/h.  fp32 contexts keep positions as the two-float sum x + xl: t = xl + d,
// x' = fl(x + t), xl' = t - (x' - x) (exact: Fast2Sum with |t| << |x|), so the state moves by d to within an ulp of d,
// not of x (rounding x_n + d to fp32 every step was the floor of the displacement error).
template <typename T>
__global__ void __launch_bounds__(256)
epilogue_kernel(BucketView bv, T inv_h, T v_max) {
  T *x = static_cast<T *>(bv.field[F_X]);
  T *v = static_cast<T *>(bv.field[F_V]);
  T *xl = static_cast<T *>(bv.field[F_XL]);                // null in fp64 contexts
  const T *d = static_cast<const T *>(bv.field[F_D]);
  const int n_pad = bv.n_pad;
  const size_t total = size_t(bv.cells) * n_pad;          // one thread per (cell, vertex slot)
  for (size_t i = blockIdx.x * size_t(blockDim.x) + threadIdx.x; i < total; i += size_t(gridDim.x) * blockDim.x) {
    const size_t base = (i / n_pad) * 3 * size_t(n_pad) + i % n_pad;
    T vi[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const size_t o = base + size_t(k) * n_pad;
      const T di = d[o];
      if (xl) {
        const T x0 = x[o], t = xl[o] + di, x1 = x0 + t;
        x[o] = x1;
        xl[o] = t - (x1 - x0);
      } else {
        x[o] += di;
      }
      vi[k] = di * inv_h;
    }
    if (v_max > T(0)) {   // vertex-velocity cap (reading R17): clamp the magnitude, keep the direction
      const T speed = sqrt(vi[0] * vi[0] + vi[1] * vi[1] + vi[2] * vi[2]);
      const T scale = speed > v_max ? v_max / speed : T(1);
#pragma unroll
      for (int k = 0; k < 3; ++k) vi[k] *= scale;
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) v[base + size_t(k) * n_pad] = vi[k];
  }
}

// fp32 fast path: one thread per 4 vertex slots, 128-bit accesses, all nine loads in flight before the stores
__global__ void __launch_bounds__(256)
epilogue_vec4_kernel(BucketView bv, float inv_h, float v_max) {
  float *x = static_cast<float *>(bv.field[F_X]);
  float *v = static_cast<float *>(bv.field[F_V]);
  float *xl = static_cast<float *>(bv.field[F_XL]);
  const float *d = static_cast<const float *>(bv.field[F_D]);
  const unsigned q_pad = unsigned(bv.n_pad) >> 2;
  const size_t total = size_t(bv.cells) * q_pad;
  for (size_t i = blockIdx.x * size_t(blockDim.x) + threadIdx.x; i < total; i += size_t(gridDim.x) * blockDim.x) {
    const size_t cell = i / q_pad;
    const size_t base = cell * 3 * size_t(bv.n_pad) + 4 * (i - cell * q_pad);
    float4 di[3], xi[3], li[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      di[k] = __ldcs(reinterpret_cast<const float4 *>(d + base + size_t(k) * bv.n_pad));
      xi[k] = *reinterpret_cast<const float4 *>(x + base + size_t(k) * bv.n_pad);
      li[k] = *reinterpret_cast<const float4 *>(xl + base + size_t(k) * bv.n_pad);
    }
    float sc[4] = {inv_h, inv_h, inv_h, inv_h};
    if (v_max > 0.f) {
      const float *dx = &di[0].x, *dy = &di[1].x, *dz = &di[2].x;
#pragma unroll
      for (int e = 0; e < 4; ++e) {   // same operations, in the same order, as the scalar kernel
        const float a = dx[e] * inv_h, b = dy[e] * inv_h, c = dz[e] * inv_h;
        const float speed = sqrtf(a * a + b * b + c * c);
        sc[e] = speed > v_max ? v_max / speed : 1.f;
      }
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const float4 dk = di[k];
      float4 xo, lo, vo;
      const float *x0 = &xi[k].x, *l0 = &li[k].x, *de = &dk.x;
      float *x1 = &xo.x, *l1 = &lo.x;
#pragma unroll
      for (int e = 0; e < 4; ++e) {   // compensated x + xl += d (see epilogue_kernel)
        const float t = l0[e] + de[e];
        x1[e] = x0[e] + t;
        l1[e] = t - (x1[e] - x0[e]);
      }
      if (v_max > 0.f) {
        vo.x = dk.x * inv_h * sc[0]; vo.y = dk.y * inv_h * sc[1]; vo.z = dk.z * inv_h * sc[2]; vo.w = dk.w * inv_h * sc[3];
      } else {
        vo.x = dk.x * inv_h; vo.y = dk.y * inv_h; vo.z = dk.z * inv_h; vo.w = dk.w * inv_h;
      }
      *reinterpret_cast<float4 *>(x + base + size_t(k) * bv.n_pad) = xo;
      *reinterpret_cast<float4 *>(xl + base + size_t(k) * bv.n_pad) = lo;
      *reinterpret_cast<float4 *>(v + base + size_t(k) * bv.n_pad) = vo;
    }
  }
}

}  // namespace

int launch_prologue(const TypeDev &td, const BucketView &bv, int precision, cudaStream_t s) {
  if (bv.cells == 0) return 0;
  const unsigned grid = unsigned(bv.cells < 148 * 16 ? bv.cells : 148 * 16);
  if (precision == NPFEM_F32 && td.n <= 32 * 21) {
    // warp per cell; 4 warps per CTA, enough CTAs to fill the machine several times over
    const int64_t ctas = (bv.cells + 3) / 4;
    const unsigned g = unsigned(ctas < 148 * 24 ? ctas : 148 * 24);
    if (td.n <= 32 * 6)
      prologue_warp_kernel<6><<<g, 128, 0, s>>>(bv, static_cast<const float *>(td.vtx_mass), float(td.kappa), float(td.h));
    else
      prologue_warp_kernel<21><<<g, 128, 0, s>>>(bv, static_cast<const float *>(td.vtx_mass), float(td.kappa), float(td.h));
  } else if (precision == NPFEM_F32)
    prologue_kernel<float><<<grid, 256, 0, s>>>(bv, static_cast<const float *>(td.vtx_mass), td.kappa, td.h);
  else
    prologue_kernel<double><<<grid, 256, 0, s>>>(bv, static_cast<const double *>(td.vtx_mass), td.kappa, td.h);
  return 1;
}

int launch_epilogue(const TypeDev &td, const BucketView &bv, int precision, double v_max, cudaStream_t s) {
  if (bv.cells == 0) return 0;
  const size_t total = size_t(bv.cells) * bv.n_pad;
  const unsigned grid = unsigned((total + 255) / 256 < 148 * 16 ? (total + 255) / 256 : 148 * 16);
  if (precision == NPFEM_F32) {
    const size_t quads = total / 4;
    const unsigned g4 = unsigned((quads + 255) / 256 < 148 * 32 ? (quads + 255) / 256 : 148 * 32);
    epilogue_vec4_kernel<<<g4, 256, 0, s>>>(bv, float(1.0 / td.h), float(v_max));
  } else
    epilogue_kernel<double><<<grid, 256, 0, s>>>(bv, 1.0 / td.h, v_max);
  return 1;
}

}  // namespace npfem
