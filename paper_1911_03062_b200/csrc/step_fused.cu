// Whole time step of one cell in ONE kernel, for the small-batch regime: the paper's
// own GPU kernel runs "the entire solver time step of one cell ... in one kernel call, one CUDA block
// per blood cell" on ~114 cells per GPU.  With so few cells the batched
// path of npfem_step (prologue, K x [local step, tensor-core GEMM], epilogue = 2 + 2K launches per
// type, each a 5-15 us kernel on a mostly idle GPU) is launch- and latency-bound.  Here one CTA takes a
// cell through prologue, K iterations and epilogue with the state in shared memory:
//   prologue  PBD damping (fp64 moments, block reduction), b = M v/h + F, d = h v
//   K times   local step = the scheduled kernel's phases (local_sched.cu: same create-time schedule,
//             same registers-resident topology, same reduced gradient r), then the global step as a
//             per-cell product  d <- (1 - gamma) d - H~^-1 r  in FP32 FFMA, H~^-1 (symmetric) streamed
//             from L2 column-wise so that the loads of a warp coalesce
//   epilogue  x_{n+1} = x_n + d, v_{n+1} = d/h, optional velocity cap
// The product reads the whole operator once per cell and iteration, so this path only pays for small
// batches; npfem_step picks it when every bucket has at most a few cells per SM (and no diagnostics,
// line search, collisions or per-kernel timing are requested).
#include "internal.h"

namespace npfem {
namespace {

__device__ __forceinline__ float rsqrt_fast(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ uint32_t lo16(uint32_t w) { return w & 0xffffu; }
__device__ __forceinline__ uint32_t hi16(uint32_t w) { return w >> 16; }
__device__ __forceinline__ float4 lds4(const unsigned char *base, uint32_t off) {
  return *reinterpret_cast<const float4 *>(base + off);
}
__device__ __forceinline__ void sts4(unsigned char *base, uint32_t off, float x, float y, float z, float w) {
  *reinterpret_cast<float4 *>(base + off) = make_float4(x, y, z, w);
}

struct FusedParams {
  int n, T, n_pad, ttri, threads, vstride, n_iterations;
  int sx_bytes, sN_bytes, sC_bytes;
  const uint32_t *tri_words;   // [TPT][5][threads]
  const float *tri_consts;     // [TPT][12][threads]
  const uint32_t *vtx_words;   // [1 + MAXV/2][vstride]
  const float *vtx_coef;       // [vstride]  (1 - gamma)(1 + h alpha) m_v / h^2
  const float *mass;           // [n]
  const float *Hinv;           // [n_pad][n_pad], symmetric
  float fx_scale;              // fixed-point volume reduction (see local_sched.cu)
  long long fx_rest;
  float vc_scale;
  float kappa, h, d_scale, v_max;
  float *x, *xl, *v;           // [cells][3][n_pad], updated; positions are the two-float sum x + xl (internal.h F_XL)
  const float *f;
  double *origin;              // [cells][3]
  int64_t cells;
};

// sum over the block of N doubles per thread; every thread gets the result
template <int N>
__device__ __forceinline__ void block_sum(double (&val)[N], double *red /* [32][N] */, int nwarps) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int k = 0; k < N; ++k)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) val[k] += __shfl_xor_sync(0xffffffffu, val[k], o);
  __syncthreads();
  if (lane == 0)
#pragma unroll
    for (int k = 0; k < N; ++k) red[warp * N + k] = val[k];
  __syncthreads();
#pragma unroll
  for (int k = 0; k < N; ++k) {
    double s = 0.0;
    for (int w = 0; w < nwarps; ++w) s += red[w * N + k];
    val[k] = s;
  }
}

template <int TPT, int MAXV>
__global__ void __launch_bounds__(256, 1) step_fused_kernel(const FusedParams p) {
  extern __shared__ __align__(16) unsigned char smem[];
  const int n = p.n, n_pad = p.n_pad, nthreads = p.threads, nwarps = nthreads >> 5;
  unsigned char *sx = smem;
  unsigned char *sN = sx + p.sx_bytes;
  unsigned char *sC = sN + p.sN_bytes;
  float *xn = reinterpret_cast<float *>(sC + p.sC_bytes);   // [3][n_pad] x_n (cell-local)
  float *sd = xn + 3 * n_pad;                               // [3][n_pad] d (v during the prologue)
  float *sb = sd + 3 * n_pad;                               // [3][n_pad] b
  float *sl = sb + 3 * n_pad;                               // [3][n_pad] low part of x_n
  float4 *sr = reinterpret_cast<float4 *>(sl + 3 * n_pad);  // [n_pad]    reduced gradient r, padding rows zero
  double *red = reinterpret_cast<double *>(sr + n_pad);     // [8][16]
  int *vacc = reinterpret_cast<int *>(red + 8 * 16);        // [2] fixed-point 6V (hi, lo)
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

  // ---- per-thread constants of the scheduled local step: registers for the whole launch ------
  uint32_t tw[TPT][5];
  float tk[TPT][12];
  bool act[TPT];
#pragma unroll
  for (int j = 0; j < TPT; ++j) {
    act[j] = tid < p.ttri && j * p.ttri + tid < p.T;
#pragma unroll
    for (int q = 0; q < 5; ++q) tw[j][q] = p.tri_words[(j * 5 + q) * nthreads + tid];
#pragma unroll
    for (int q = 0; q < 12; ++q) tk[j][q] = p.tri_consts[(j * 12 + q) * nthreads + tid];
  }
  if (tid < 8) sts4(sC, uint32_t(p.sC_bytes) - 128u + 16u * tid, 0.f, 0.f, 0.f, 0.f);   // the zero slots
  for (int i = n + tid; i < n_pad; i += nthreads) sr[i] = make_float4(0.f, 0.f, 0.f, 0.f);
  const float inv_h = 1.f / p.h;

  for (int64_t cell = blockIdx.x; cell < p.cells; cell += gridDim.x) {
    const size_t base = size_t(cell) * 3 * n_pad;
    float *xg = p.x + base, *lg = p.xl + base, *vg = p.v + base;
    const float *fg = p.f + base;
    // ================= prologue: PBD damping, b, d0 =================================================
    double s[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) s[k] = 0.0;
    for (int i = tid; i < n; i += nthreads) {
      const float x0f = xg[i], x1f = xg[n_pad + i], x2f = xg[2 * n_pad + i];
      const float v0f = vg[i], v1f = vg[n_pad + i], v2f = vg[2 * n_pad + i];
      xn[i] = x0f; xn[n_pad + i] = x1f; xn[2 * n_pad + i] = x2f;
      sl[i] = lg[i]; sl[n_pad + i] = lg[n_pad + i]; sl[2 * n_pad + i] = lg[2 * n_pad + i];
      sd[i] = v0f; sd[n_pad + i] = v1f; sd[2 * n_pad + i] = v2f;
      const double md = double(p.mass[i]);
      const double x0 = x0f, x1 = x1f, x2 = x2f, p0 = md * v0f, p1 = md * v1f, p2 = md * v2f;
      s[0] += md;
      s[1] += md * x0; s[2] += md * x1; s[3] += md * x2;
      s[4] += p0; s[5] += p1; s[6] += p2;
      s[7] += x1 * p2 - x2 * p1; s[8] += x2 * p0 - x0 * p2; s[9] += x0 * p1 - x1 * p0;
      s[10] += md * x0 * x0; s[11] += md * x1 * x1; s[12] += md * x2 * x2;
      s[13] += md * x0 * x1; s[14] += md * x0 * x2; s[15] += md * x1 * x2;
    }
    block_sum<16>(s, red, nwarps);
    const double M = s[0], inv_M = 1.0 / M;
    const double xc[3] = {s[1] * inv_M, s[2] * inv_M, s[3] * inv_M};
    const double vc3[3] = {s[4] * inv_M, s[5] * inv_M, s[6] * inv_M};
    double om[3] = {0.0, 0.0, 0.0};
    if (p.kappa > 0.f) {   // about the mass centre: L_c = L_0 - x_c x P,  S_c = S_0 - M x_c x_c^T
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
    float shift[3] = {0.f, 0.f, 0.f};
    const bool recentre = fabs(xc[0]) > 0.5 || fabs(xc[1]) > 0.5 || fabs(xc[2]) > 0.5;
    if (recentre) {   // exact binary shift of the local frame, as in prologue.cu
      double sh[3];
#pragma unroll
      for (int k = 0; k < 3; ++k) { sh[k] = rint(xc[k] * 1024.0) / 1024.0; shift[k] = float(sh[k]); }
      if (tid < 3) p.origin[size_t(cell) * 3 + tid] += tid == 0 ? sh[0] : (tid == 1 ? sh[1] : sh[2]);
    }
    const float xcf[3] = {float(xc[0]), float(xc[1]), float(xc[2])}, vcf[3] = {float(vc3[0]), float(vc3[1]), float(vc3[2])};
    const float omf[3] = {float(om[0]), float(om[1]), float(om[2])};
    for (int i = tid; i < n; i += nthreads) {
      float xi[3] = {xn[i], xn[n_pad + i], xn[2 * n_pad + i]};
      float vi[3] = {sd[i], sd[n_pad + i], sd[2 * n_pad + i]};
      if (p.kappa > 0.f) {
        const float r0 = xi[0] - xcf[0], r1 = xi[1] - xcf[1], r2 = xi[2] - xcf[2];
        const float w[3] = {omf[1] * r2 - omf[2] * r1, omf[2] * r0 - omf[0] * r2, omf[0] * r1 - omf[1] * r0};
#pragma unroll
        for (int k = 0; k < 3; ++k) vi[k] += p.kappa * (vcf[k] + w[k] - vi[k]);
      }
      const float mh = p.mass[i] * inv_h;
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        if (recentre) {   // rare; the rounding of the shifted coordinate goes to the low part
          const double xs = double(xi[k]) - double(shift[k]);
          const float hi = float(xs);
          xn[k * n_pad + i] = hi;
          sl[k * n_pad + i] += float(xs - double(hi));
        }
        sb[k * n_pad + i] = fmaf(mh, vi[k], fg[k * n_pad + i]);
        sd[k * n_pad + i] = p.h * vi[k];
      }
    }
    __syncthreads();
    // ================= K quasi-Newton iterations =====================================================
    for (int k_it = 0; k_it < p.n_iterations; ++k_it) {
      // ---- phase 0: sx[slot(v)] = (x_n + d, 0) ---------------------------------------------------
      for (int i = tid; i < n; i += nthreads)
        sts4(sx, lo16(p.vtx_words[i]), xn[i] + (sl[i] + sd[i]), xn[n_pad + i] + (sl[n_pad + i] + sd[n_pad + i]),
             xn[2 * n_pad + i] + (sl[2 * n_pad + i] + sd[2 * n_pad + i]), 0.f);
      if (tid == 0) vacc[0] = vacc[1] = 0;
      if (tid < 8) sts4(sC, uint32_t(p.sC_bytes) - 128u + 16u * tid, 0.f, 0.f, 0.f, 0.f);   // the zero slots (sC doubles as scratch)
      __syncthreads();
      // ---- phase A: edges, unit normal, volume partial ----------------------------------------------
      float e1[TPT][3], e2[TPT][3], nh[TPT][3], inv[TPT], nn[TPT];
      float vol = 0.f;
#pragma unroll
      for (int j = 0; j < TPT; ++j) {
        const float4 X0 = lds4(sx, lo16(tw[j][0])), X1 = lds4(sx, hi16(tw[j][0])), X2 = lds4(sx, lo16(tw[j][1]));
        e1[j][0] = X1.x - X0.x; e1[j][1] = X1.y - X0.y; e1[j][2] = X1.z - X0.z;
        e2[j][0] = X2.x - X0.x; e2[j][1] = X2.y - X0.y; e2[j][2] = X2.z - X0.z;
        const float Nx = e1[j][1] * e2[j][2] - e1[j][2] * e2[j][1];
        const float Ny = e1[j][2] * e2[j][0] - e1[j][0] * e2[j][2];
        const float Nz = e1[j][0] * e2[j][1] - e1[j][1] * e2[j][0];
        nn[j] = Nx * Nx + Ny * Ny + Nz * Nz;
        vol += act[j] ? X0.x * Nx + X0.y * Ny + X0.z * Nz : 0.f;
        inv[j] = rsqrt_fast(nn[j]);
        nh[j][0] = Nx * inv[j]; nh[j][1] = Ny * inv[j]; nh[j][2] = Nz * inv[j];
        if (act[j]) sts4(sN, hi16(tw[j][4]), nh[j][0], nh[j][1], nh[j][2], inv[j]);
      }
      {
        const int wsum = __reduce_add_sync(0xffffffffu, __float2int_rn(vol * p.fx_scale));
        if (lane == 0) {
          atomicAdd(vacc, wsum >> 12);
          atomicAdd(vacc + 1, wsum & 0xfff);
        }
      }
      // membrane (Skalak, readings R5/R7): Q = 2 A0 (W1 R + W2 det^2 adj G)
      float e11[TPT], e12[TPT], e22[TPT], q11[TPT], q12[TPT], q22[TPT];
#pragma unroll
      for (int j = 0; j < TPT; ++j) {
        const float *a1 = e1[j], *a2 = e2[j];
        e11[j] = a1[0] * a1[0] + a1[1] * a1[1] + a1[2] * a1[2];
        e12[j] = a1[0] * a2[0] + a1[1] * a2[1] + a1[2] * a2[2];
        e22[j] = a2[0] * a2[0] + a2[1] * a2[1] + a2[2] * a2[2];
        const float R11 = tk[j][0], R12 = tk[j][1], R22 = tk[j][2], J = tk[j][3], tA = tk[j][4], tC = tk[j][5];
        const float th = fmaf(R12, e12[j], -0.5f);
        const float I1p1 = fmaf(R11, e11[j], fmaf(R22, e22[j], th + th));
        const float I2 = fmaf(J, nn[j], -1.f);
        const float W1 = tA * I1p1, W2 = fmaf(tC, I2, -tA * J);
        q11[j] = fmaf(W2, e22[j], W1 * R11);
        q22[j] = fmaf(W2, e11[j], W1 * R22);
        q12[j] = fmaf(-W2, e12[j], W1 * R12);
      }
      __syncthreads();                                   // sN complete, volume accumulated
      // ---- phase B: hinges (reading R8), volume term (R9), corner forces -------------------------------
      // (the cast to int is the modular reduction of the wrapped int32 sums: see local_sched.cu for the validity range)
      const float vc = p.vc_scale * float(int((static_cast<long long>(vacc[0]) << 12) + vacc[1] - p.fx_rest));
#pragma unroll
      for (int j = 0; j < TPT; ++j) {
        const float *a1 = e1[j], *a2 = e2[j], *nA = nh[j];
        const float4 NB0 = lds4(sN, hi16(tw[j][1])), NB1 = lds4(sN, lo16(tw[j][2])), NB2 = lds4(sN, hi16(tw[j][2]));
        float w0 = 0.f, w1 = 0.f, w2 = 0.f;
        {
          const float4 B = NB0;
          const float crx = nA[1] * B.z - nA[2] * B.y, cry = nA[2] * B.x - nA[0] * B.z, crz = nA[0] * B.y - nA[1] * B.x;
          const float S = crx * a1[0] + cry * a1[1] + crz * a1[2];
          const float cs = nA[0] * B.x + nA[1] * B.y + nA[2] * B.z;
          const float L = e11[j], D = e11[j] - e12[j], ie = rsqrt_fast(L);
          const float q = ie * fmaf(S * ie, tk[j][6], -cs * tk[j][9]);
          w0 = fmaf(D, q, w0); w1 = fmaf(L - D, q, w1); w2 = fmaf(-L, q, w2);
        }
        {
          const float4 B = NB1;
          const float crx = nA[1] * B.z - nA[2] * B.y, cry = nA[2] * B.x - nA[0] * B.z, crz = nA[0] * B.y - nA[1] * B.x;
          const float S = crx * (a2[0] - a1[0]) + cry * (a2[1] - a1[1]) + crz * (a2[2] - a1[2]);
          const float cs = nA[0] * B.x + nA[1] * B.y + nA[2] * B.z;
          const float L = e11[j] - 2.f * e12[j] + e22[j], D = e22[j] - e12[j], ie = rsqrt_fast(L);
          const float q = ie * fmaf(S * ie, tk[j][7], -cs * tk[j][10]);
          w1 = fmaf(D, q, w1); w2 = fmaf(L - D, q, w2); w0 = fmaf(-L, q, w0);
        }
        {
          const float4 B = NB2;
          const float crx = nA[1] * B.z - nA[2] * B.y, cry = nA[2] * B.x - nA[0] * B.z, crz = nA[0] * B.y - nA[1] * B.x;
          const float S = -(crx * a2[0] + cry * a2[1] + crz * a2[2]);
          const float cs = nA[0] * B.x + nA[1] * B.y + nA[2] * B.z;
          const float L = e22[j], D = e12[j], ie = rsqrt_fast(L);
          const float q = ie * fmaf(S * ie, tk[j][8], -cs * tk[j][11]);
          w2 = fmaf(D, q, w2); w0 = fmaf(L - D, q, w0); w1 = fmaf(-L, q, w1);
        }
        const float vn = vc * (nn[j] * inv[j]);
        const float u0 = fmaf(inv[j], w0, vn), u1 = fmaf(inv[j], w1, vn), u2 = fmaf(inv[j], w2, vn);
        const float us = u0 + u1 + u2;
        float c0[3], c1[3], c2[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
          c1[k] = fmaf(u1, nA[k], fmaf(q11[j], a1[k], q12[j] * a2[k]));
          c2[k] = fmaf(u2, nA[k], fmaf(q12[j], a1[k], q22[j] * a2[k]));
          c0[k] = fmaf(us, nA[k], -c1[k]) - c2[k];
        }
        if (act[j]) {
          sts4(sC, lo16(tw[j][3]), c0[0], c0[1], c0[2], 0.f);
          sts4(sC, hi16(tw[j][3]), c1[0], c1[1], c1[2], 0.f);
          sts4(sC, lo16(tw[j][4]), c2[0], c2[1], c2[2], 0.f);
        }
      }
      __syncthreads();                                   // corner forces complete
      // ---- phase C: r = coef d - b + sum of the vertex's corner forces -> sr -----------------------
      for (int i = tid; i < n; i += nthreads) {
        float ax = 0.f, ay = 0.f, az = 0.f;
#pragma unroll
        for (int q = 0; q < MAXV / 2; ++q) {
          const uint32_t w = p.vtx_words[(1 + q) * p.vstride + i];
          const float4 fa = lds4(sC, lo16(w)), fb = lds4(sC, hi16(w));
          ax += fa.x + fb.x; ay += fa.y + fb.y; az += fa.z + fb.z;
        }
        const float coef = p.vtx_coef[i];
        sr[i] = make_float4(fmaf(coef, sd[i], ax - sb[i]), fmaf(coef, sd[n_pad + i], ay - sb[n_pad + i]),
                            fmaf(coef, sd[2 * n_pad + i], az - sb[2 * n_pad + i]), 0.f);
      }
      __syncthreads();                                   // r complete
      // ---- global step of this cell: d <- d_scale d - H~^-1 r  (Eq. 4).  H~^-1 is symmetric: thread
      // (q, sl) accumulates rows 4q .. 4q+3 over the j of its slice from 128-bit loads of row j (= column j),
      // r_j is a shared-memory broadcast; the slices' partial sums meet in shared memory (the corner-force
      // buffer is free here) ----------------------------------------------------------------------------
      {
        const int nq = n_pad >> 2;                        // row quads (n_pad is a multiple of 16)
        int slices = nthreads / nq;
        const int cap = p.sC_bytes / (n_pad * 16);
        slices = slices < cap ? slices : cap;             // >= 1 for every supported type (checked on the host)
        const int q = tid % nq, sl = tid / nq;
        float4 *part = reinterpret_cast<float4 *>(sC);    // [slices][n_pad] (u0, u1, u2, -) of row i
        if (sl < slices) {
          float u[4][3];
#pragma unroll
          for (int r4 = 0; r4 < 4; ++r4) u[r4][0] = u[r4][1] = u[r4][2] = 0.f;
          const int per = (n + slices - 1) / slices, j0 = sl * per, j1 = min(n, j0 + per);
          const float4 *col = reinterpret_cast<const float4 *>(p.Hinv) + q;
#pragma unroll 8
          for (int j = j0; j < j1; ++j) {
            const float4 w = __ldg(col + size_t(j) * nq);
            const float4 r = sr[j];
            u[0][0] = fmaf(w.x, r.x, u[0][0]); u[0][1] = fmaf(w.x, r.y, u[0][1]); u[0][2] = fmaf(w.x, r.z, u[0][2]);
            u[1][0] = fmaf(w.y, r.x, u[1][0]); u[1][1] = fmaf(w.y, r.y, u[1][1]); u[1][2] = fmaf(w.y, r.z, u[1][2]);
            u[2][0] = fmaf(w.z, r.x, u[2][0]); u[2][1] = fmaf(w.z, r.y, u[2][1]); u[2][2] = fmaf(w.z, r.z, u[2][2]);
            u[3][0] = fmaf(w.w, r.x, u[3][0]); u[3][1] = fmaf(w.w, r.y, u[3][1]); u[3][2] = fmaf(w.w, r.z, u[3][2]);
          }
#pragma unroll
          for (int r4 = 0; r4 < 4; ++r4) part[sl * n_pad + 4 * q + r4] = make_float4(u[r4][0], u[r4][1], u[r4][2], 0.f);
        }
        __syncthreads();                                  // partial sums complete
        for (int i = tid; i < n; i += nthreads) {
          float u0 = 0.f, u1 = 0.f, u2 = 0.f;
          for (int s2 = 0; s2 < slices; ++s2) {
            const float4 v4 = part[s2 * n_pad + i];
            u0 += v4.x; u1 += v4.y; u2 += v4.z;
          }
          sd[i] = fmaf(p.d_scale, sd[i], -u0);
          sd[n_pad + i] = fmaf(p.d_scale, sd[n_pad + i], -u1);
          sd[2 * n_pad + i] = fmaf(p.d_scale, sd[2 * n_pad + i], -u2);
        }
      }
      __syncthreads();                                   // d complete
    }
    // ================= epilogue: x_{n+1} = x_n + d, v_{n+1} = d / h (Eq. 1), velocity cap ================
    for (int i = tid; i < n; i += nthreads) {
      float vi[3];
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        const float di = sd[k * n_pad + i];
        const float x0 = xn[k * n_pad + i], t = sl[k * n_pad + i] + di, x1 = x0 + t;   // compensated x + xl += d (prologue.cu)
        xg[k * n_pad + i] = x1;
        lg[k * n_pad + i] = t - (x1 - x0);
        vi[k] = di * inv_h;
      }
      if (p.v_max > 0.f) {
        const float speed = sqrtf(vi[0] * vi[0] + vi[1] * vi[1] + vi[2] * vi[2]);
        const float scale = speed > p.v_max ? p.v_max / speed : 1.f;
#pragma unroll
        for (int k = 0; k < 3; ++k) vi[k] *= scale;
      }
#pragma unroll
      for (int k = 0; k < 3; ++k) vg[k * n_pad + i] = vi[k];
    }
    __syncthreads();                                     // shared memory is reused by the next cell
  }
}

size_t fused_smem_bytes(const SchedDev &s, int n_pad) {
  return size_t(s.n_vslots + s.n_tslots + s.n_cslots) * 16 + size_t(12) * n_pad * 4 + size_t(n_pad) * 16 + 8 * 16 * 8 + 16;
}

}  // namespace

bool step_fused_supported(const TypeDev &td) {
  const SchedDev &s = td.sched;
  return s.valid && s.threads <= 256 && td.Hinv != nullptr && fused_smem_bytes(s, td.n_pad) <= 200 * 1024 &&
         td.n_pad / 4 <= s.threads && s.n_cslots * 16 >= td.n_pad * 16;
}

int launch_step_fused(const TypeDev &td, const BucketView &bv, int n_sm, int n_iterations, double v_max, cudaStream_t stream) {
  if (bv.cells == 0) return 0;
  if (!step_fused_supported(td)) return -1;
  const SchedDev &s = td.sched;
  FusedParams p;
  p.n = td.n; p.T = td.T; p.n_pad = td.n_pad; p.ttri = s.ttri; p.threads = s.threads; p.vstride = s.vstride;
  p.n_iterations = n_iterations;
  p.sx_bytes = s.n_vslots * 16; p.sN_bytes = s.n_tslots * 16; p.sC_bytes = s.n_cslots * 16;
  p.tri_words = s.tri_words; p.tri_consts = s.tri_consts; p.vtx_words = s.vtx_words; p.vtx_coef = s.vtx_coef;
  p.mass = static_cast<const float *>(td.vtx_mass);
  p.Hinv = static_cast<const float *>(td.Hinv);
  int k = 0;
  std::frexp(16.0 * 32.0 * s.vol_lane_bound, &k);   // same fixed-point scale as local_sched.cu
  const double scale = std::ldexp(1.0, 31 - k);
  p.fx_scale = float(scale);
  p.fx_rest = std::llrint(6.0 * td.V0 * scale);
  p.vc_scale = float(td.kv_over_V0 / 36.0 / scale);
  p.kappa = float(td.kappa); p.h = float(td.h); p.d_scale = float(1.0 - td.gamma); p.v_max = float(v_max);
  p.x = static_cast<float *>(bv.field[F_X]);
  p.xl = static_cast<float *>(bv.field[F_XL]);
  p.v = static_cast<float *>(bv.field[F_V]);
  p.f = static_cast<const float *>(bv.field[F_F]);
  p.origin = bv.origin;
  p.cells = bv.cells;
  const size_t smem = fused_smem_bytes(s, td.n_pad);
  auto launch = [&](auto kernel) -> int {
    if (!td.cache.fused_attr) {   // per context and type (the attribute is per device)
      if (opt_in_max_dynamic_smem(kernel) != cudaSuccess) return -1;
      td.cache.fused_attr = true;
    }
    const int64_t grid = bv.cells < int64_t(n_sm) * 4 ? bv.cells : int64_t(n_sm) * 4;
    kernel<<<unsigned(grid), s.threads, smem, stream>>>(p);
    return 1;
  };
  if (s.tpt == 2) return s.maxv == 6 ? launch(step_fused_kernel<2, 6>) : launch(step_fused_kernel<2, 8>);
  return s.maxv == 6 ? launch(step_fused_kernel<1, 6>) : launch(step_fused_kernel<1, 8>);
}

}  // namespace npfem
