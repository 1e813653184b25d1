// Local step (row a2), generic kernel for any mesh size and both precisions, and the objective
// diagnostic (row a5).
//
//   g = M~ d/h^2 - b + grad E(x_n + d),   E = E_strain + E_area + E_bend + E_vol
//   (grad g of Eq. (3)/(4), written in the displacement d = x - x_n;
//    F_int = -grad E; energies per readings R5-R9)
//
// One CTA works on one cell at a time (cells are independent).  The cell's current
// positions are staged in shared memory; the work is TRIANGLE-CENTRIC:
//   phase A  per triangle: area vector N_t = e1 x e2 (kept for the neighbours), volume partial;
//            per vertex : first one-ring pass of the Rayleigh operator, z = k_mem d + k_b (L_cot d)/A_v
//   phase B  per triangle: Skalak membrane gradient, and for each of its 3 edges the hinge
//            gradient restricted to THIS triangle's corners - every hinge force on a vertex is a
//            multiple of the area vector of one of the two triangles, so each triangle only needs
//            its neighbour's N.  The volume gradient of a closed surface is (1/6) sum_{t in ring} N_t
//            and rides on the same corner slots.  9 numbers per triangle -> corner buffer.
//   phase C  per vertex: gather its <= valence_max corner slots in a fixed order (deterministic,
//            no atomics), add the inertia + Rayleigh stencil and -b, write g coalesced.
#include "internal.h"

namespace npfem {

template <typename T>
struct LocalParams {
  int n, T_, n_pad, valence_max;
  const int4 *tri, *tri_nbr;
  const T *tri_rest, *hinge_rest;
  const int *vtx_corner, *vtx_nbr;
  const T *vtx_w, *vtx_mass, *vtx_inv_area;
  T B4, C4, k_b, kv_over_V0, V0, k_mem, beta_over_h, inertia_coef;
  const T *x, *xl, *d, *b;   // xl: low part of the two-float positions of fp32 contexts (internal.h F_XL), else null
  T *g;
  int64_t cells;
  T *scratch;          // global scratch per CTA when the working set does not fit in shared memory:
  int g_tf32;          // round g to TF32 (fp32 contexts whose global step runs on the tensor cores)
  int scratch_in_smem; //   1: nothing, 0: [13 T_] normals + corner forces, -1: [9 n + 13 T_] the vertex arrays too
};

namespace {

__device__ __forceinline__ void cross3(const double *u, const double *v, double *w) {
  w[0] = u[1] * v[2] - u[2] * v[1];
  w[1] = u[2] * v[0] - u[0] * v[2];
  w[2] = u[0] * v[1] - u[1] * v[0];
}
__device__ __forceinline__ double dot3(const double *u, const double *v) {
  return u[0] * v[0] + u[1] * v[1] + u[2] * v[2];
}
__device__ __forceinline__ float rsq(float x) { return rsqrtf(x); }
__device__ __forceinline__ double rsq(double x) { return rsqrt(x); }

template <typename T, int NT>
__global__ void __launch_bounds__(NT, NT == 256 ? 2 : 1)
local_generic_kernel(const LocalParams<T> p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ double red[16];
  __shared__ T vol_coef_sh;
  const int n = p.n, n_pad = p.n_pad, nt = p.T_;
  // any mesh size runs: what does not fit in shared memory lives in a per-CTA slab of global scratch
  // (L2-resident; __syncthreads orders global accesses within the block as well)
  T *slab = p.scratch_in_smem > 0 ? nullptr
                                  : p.scratch + size_t(blockIdx.x) * (p.scratch_in_smem < 0 ? size_t(9) * n + size_t(13) * nt : size_t(13) * nt);
  T *sx = p.scratch_in_smem < 0 ? slab : reinterpret_cast<T *>(smem_raw);   // [3][n] current positions x_n + d (cell-local)
  T *sd = sx + 3 * n;                        // [3][n] d
  T *sz = sd + 3 * n;                        // [3][n] z
  T *sN, *sC;
  if (p.scratch_in_smem > 0) {
    sN = sz + 3 * n;                         // [T][4] area vector, |N|^2
    sC = sN + 4 * nt;                        // [T][9] corner forces
  } else {
    sN = p.scratch_in_smem < 0 ? sz + 3 * n : slab;
    sC = sN + 4 * nt;
  }
  const bool stencil = p.beta_over_h != T(0);

  for (int64_t cell = blockIdx.x; cell < p.cells; cell += gridDim.x) {
    const size_t base = size_t(cell) * 3 * n_pad;
    // ---- phase 0: stage x = x_n + d and d ---------------------------------------------------
    for (int k = 0; k < 3; ++k)
      for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const T dd = p.d[base + k * n_pad + i];
        sx[k * n + i] = p.x[base + k * n_pad + i] + (p.xl ? p.xl[base + k * n_pad + i] + dd : dd);
        sd[k * n + i] = dd;
      }
    __syncthreads();
    // ---- phase A ----------------------------------------------------------------------------
    double vol = 0.0;
    for (int t = threadIdx.x; t < nt; t += blockDim.x) {
      const int4 tv = p.tri[t];
      const T x0[3] = {sx[tv.x], sx[n + tv.x], sx[2 * n + tv.x]};
      const T e1[3] = {sx[tv.y] - x0[0], sx[n + tv.y] - x0[1], sx[2 * n + tv.y] - x0[2]};
      const T e2[3] = {sx[tv.z] - x0[0], sx[n + tv.z] - x0[1], sx[2 * n + tv.z] - x0[2]};
      const T N0 = e1[1] * e2[2] - e1[2] * e2[1];
      const T N1 = e1[2] * e2[0] - e1[0] * e2[2];
      const T N2 = e1[0] * e2[1] - e1[1] * e2[0];
      sN[4 * t + 0] = N0;
      sN[4 * t + 1] = N1;
      sN[4 * t + 2] = N2;
      sN[4 * t + 3] = N0 * N0 + N1 * N1 + N2 * N2;
      vol += double(x0[0] * N0 + x0[1] * N1 + x0[2] * N2);
    }
    if (stencil)
      for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const T w0 = p.vtx_w[i];
        T u[3] = {w0 * sd[i], w0 * sd[n + i], w0 * sd[2 * n + i]};
        for (int q = 0; q < p.valence_max; ++q) {
          const int j = p.vtx_nbr[q * n + i];
          const T w = p.vtx_w[(q + 1) * n + i];
          u[0] += w * sd[j];
          u[1] += w * sd[n + j];
          u[2] += w * sd[2 * n + j];
        }
        const T s = p.k_b * p.vtx_inv_area[i];
        for (int k = 0; k < 3; ++k) sz[k * n + i] = p.k_mem * sd[k * n + i] + s * u[k];
      }
    // block reduction of the volume (also orders phase A before phase B)
    for (int o = 16; o > 0; o >>= 1) vol += __shfl_xor_sync(0xffffffffu, vol, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = vol;
    __syncthreads();
    if (threadIdx.x == 0) {
      double s = 0.0;
      for (int i = 0; i < int(blockDim.x >> 5); ++i) s += red[i];
      const double V = s / 6.0;
      vol_coef_sh = T(double(p.kv_over_V0) * (V - double(p.V0)) / 6.0);   // k_v (V - V0)/V0 / 6
    }
    __syncthreads();
    const T vol_coef = vol_coef_sh;
    // ---- phase B ----------------------------------------------------------------------------
    for (int t = threadIdx.x; t < nt; t += blockDim.x) {
      const int4 tv = p.tri[t];
      const int4 tn = p.tri_nbr[t];
      const T a = p.tri_rest[4 * t], b = p.tri_rest[4 * t + 1], c = p.tri_rest[4 * t + 2], A0 = p.tri_rest[4 * t + 3];
      const T x0[3] = {sx[tv.x], sx[n + tv.x], sx[2 * n + tv.x]};
      const T e1[3] = {sx[tv.y] - x0[0], sx[n + tv.y] - x0[1], sx[2 * n + tv.y] - x0[2]};
      const T e2[3] = {sx[tv.z] - x0[0], sx[n + tv.z] - x0[1], sx[2 * n + tv.z] - x0[2]};
      const T NA[3] = {sN[4 * t], sN[4 * t + 1], sN[4 * t + 2]};
      const T nnA = sN[4 * t + 3];
      const T e11 = e1[0] * e1[0] + e1[1] * e1[1] + e1[2] * e1[2];
      const T e12 = e1[0] * e2[0] + e1[1] * e2[1] + e1[2] * e2[2];
      const T e22 = e2[0] * e2[0] + e2[1] * e2[1] + e2[2] * e2[2];
      // membrane: F = [a e1, b e1 + c e2], C = F^T F
      const T C11 = a * a * e11;
      const T C12 = a * (b * e11 + c * e12);
      const T C22 = b * b * e11 + T(2) * b * c * e12 + c * c * e22;
      const T I1 = C11 + C22 - T(2);
      const T I2 = C11 * C22 - C12 * C12 - T(1);
      const T W1 = p.B4 * (I1 + T(1));
      const T W2 = p.C4 * I2 - p.B4;
      const T S11 = T(2) * (W1 + W2 * C22), S12 = T(-2) * W2 * C12, S22 = T(2) * (W1 + W2 * C11);
      // P = F S = [p11 e1 + p12 e2, p21 e1 + p22 e2];  [g1 g2] = A0 P Dm^-T = A0 [a P1 + b P2, c P2]
      const T p11 = S11 * a + S12 * b, p12 = S12 * c, p21 = S12 * a + S22 * b, p22 = S22 * c;
      const T al1 = A0 * (a * p11 + b * p21), al2 = A0 * (a * p12 + b * p22);
      const T be1 = A0 * c * p21, be2 = A0 * c * p22;
      T w[3] = {vol_coef, vol_coef, vol_coef};   // coefficient of N_A on corner 0, 1, 2
      // hinges: edge s runs from corner s to corner s+1, opposite corner s+2
      //   |e_0|^2 = e11, |e_1|^2 = e11 - 2 e12 + e22, |e_2|^2 = e22
      //   (x_j - x_k).e and (x_k - x_i).e in terms of e11, e12, e22
      const int nb[3] = {tn.x, tn.y, tn.z};
      const T es[3][3] = {{e1[0], e1[1], e1[2]},
                          {e2[0] - e1[0], e2[1] - e1[1], e2[2] - e1[2]},
                          {-e2[0], -e2[1], -e2[2]}};
      const T len2[3] = {e11, e11 - T(2) * e12 + e22, e22};
      const T djk[3] = {e11 - e12, e22 - e12, e12};   // (x_j - x_k).e for s = 0, 1, 2
      for (int s = 0; s < 3; ++s) {
        const T NB[3] = {sN[4 * nb[s]], sN[4 * nb[s] + 1], sN[4 * nb[s] + 2]};
        const T nnB = sN[4 * nb[s] + 3];
        const T cr0 = NA[1] * NB[2] - NA[2] * NB[1];
        const T cr1 = NA[2] * NB[0] - NA[0] * NB[2];
        const T cr2 = NA[0] * NB[1] - NA[1] * NB[0];
        const T inv_e = rsq(len2[s]);
        const T inv_nn = rsq(nnA * nnB);
        const T sin_t = (cr0 * es[s][0] + cr1 * es[s][1] + cr2 * es[s][2]) * inv_e * inv_nn;
        const T cos_t = (NA[0] * NB[0] + NA[1] * NB[1] + NA[2] * NB[2]) * inv_nn;
        const T c0 = p.hinge_rest[6 * t + 2 * s], s0 = p.hinge_rest[6 * t + 2 * s + 1];
        const T dE = p.k_b * (sin_t * c0 - cos_t * s0);      // k_b sin(theta - theta0)
        const T common = dE * inv_e / nnA;                   // dE / (|e| |N_A|^2)
        w[s] += djk[s] * common;                             // corner i = s
        w[(s + 1) % 3] += (len2[s] - djk[s]) * common;       // corner j = s+1: (x_k - x_i).e
        w[(s + 2) % 3] -= len2[s] * common;                  // corner k = s+2: -|e|/|N_A|^2
      }
      for (int k = 0; k < 3; ++k) {
        const T g1 = al1 * e1[k] + al2 * e2[k];
        const T g2 = be1 * e1[k] + be2 * e2[k];
        sC[9 * t + 0 + k] = -(g1 + g2) + w[0] * NA[k];
        sC[9 * t + 3 + k] = g1 + w[1] * NA[k];
        sC[9 * t + 6 + k] = g2 + w[2] * NA[k];
      }
    }
    __syncthreads();
    // ---- phase C ----------------------------------------------------------------------------
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
      T acc[3] = {T(0), T(0), T(0)};
      for (int q = 0; q < p.valence_max; ++q) {
        const int cid = p.vtx_corner[q * n + i];
        if (cid >= 0) {
          acc[0] += sC[3 * cid];
          acc[1] += sC[3 * cid + 1];
          acc[2] += sC[3 * cid + 2];
        }
      }
      const T mi = p.inertia_coef * p.vtx_mass[i];
      T lz[3] = {T(0), T(0), T(0)};
      if (stencil) {
        const T w0 = p.vtx_w[i];
        for (int k = 0; k < 3; ++k) lz[k] = w0 * sz[k * n + i];
        for (int q = 0; q < p.valence_max; ++q) {
          const int j = p.vtx_nbr[q * n + i];
          const T wq = p.vtx_w[(q + 1) * n + i];
          for (int k = 0; k < 3; ++k) lz[k] += wq * sz[k * n + j];
        }
      }
      for (int k = 0; k < 3; ++k) {
        const T gk = mi * sd[k * n + i] + p.beta_over_h * lz[k] - p.b[base + k * n_pad + i] + acc[k];
        p.g[base + k * n_pad + i] = p.g_tf32 ? tf32_rn(gk) : gk;
      }
    }
    __syncthreads();
  }
}

// ---- objective (row a5): fp64 arithmetic on the stored state, one CTA per cell --------------
template <typename T>
__global__ void __launch_bounds__(256)
objective_kernel(const LocalParams<T> p, const int64_t *__restrict__ cell_id, double *__restrict__ out_row,
                 const int *__restrict__ skip, double h) {
  // cell_id == nullptr: out_row is indexed by the bucket slot; skip[slot] != 0: leave that cell alone
  __shared__ double red[8];
  const int n = p.n, n_pad = p.n_pad, nt = p.T_;
  if (skip && skip[p.cells] == 0) return;               // line search: skip[cells] = cells still searching
  for (int64_t cell = blockIdx.x; cell < p.cells; cell += gridDim.x) {
    if (skip && skip[cell]) continue;
    const size_t base = size_t(cell) * 3 * n_pad;
    auto pos = [&](int v, int k) {
      return double(p.x[base + k * n_pad + v]) + ((p.xl ? double(p.xl[base + k * n_pad + v]) : 0.0) + double(p.d[base + k * n_pad + v]));
    };
    double acc = 0.0, vol = 0.0;
    for (int t = threadIdx.x; t < nt; t += blockDim.x) {
      const int4 tv = p.tri[t];
      const int4 tn = p.tri_nbr[t];
      double x0[3], e1[3], e2[3], N[3];
      for (int k = 0; k < 3; ++k) {
        x0[k] = pos(tv.x, k);
        e1[k] = pos(tv.y, k) - x0[k];
        e2[k] = pos(tv.z, k) - x0[k];
      }
      cross3(e1, e2, N);
      vol += dot3(x0, N);
      const double a = p.tri_rest[4 * t], b = p.tri_rest[4 * t + 1], c = p.tri_rest[4 * t + 2], A0 = p.tri_rest[4 * t + 3];
      const double e11 = dot3(e1, e1), e12 = dot3(e1, e2), e22 = dot3(e2, e2);
      const double C11 = a * a * e11, C12 = a * (b * e11 + c * e12), C22 = b * b * e11 + 2 * b * c * e12 + c * c * e22;
      const double I1 = C11 + C22 - 2.0, I2 = C11 * C22 - C12 * C12 - 1.0;
      acc += A0 * (double(p.B4) * (0.5 * I1 * I1 + I1 - I2) + 0.5 * double(p.C4) * I2 * I2);
      const int nb[3] = {tn.x, tn.y, tn.z};
      const int vs[3] = {tv.x, tv.y, tv.z};
      for (int s = 0; s < 3; ++s) {   // every hinge is seen from both of its triangles: half each
        const int4 tb = p.tri[nb[s]];
        double y0[3], f1[3], f2[3], NB[3], e[3], cr[3];
        for (int k = 0; k < 3; ++k) {
          y0[k] = pos(tb.x, k);
          f1[k] = pos(tb.y, k) - y0[k];
          f2[k] = pos(tb.z, k) - y0[k];
          e[k] = pos(vs[(s + 1) % 3], k) - pos(vs[s], k);
        }
        cross3(f1, f2, NB);
        cross3(N, NB, cr);
        const double inv = 1.0 / sqrt(dot3(N, N) * dot3(NB, NB));
        const double sin_t = dot3(cr, e) / sqrt(dot3(e, e)) * inv, cos_t = dot3(N, NB) * inv;
        const double c0 = p.hinge_rest[6 * t + 2 * s], s0 = p.hinge_rest[6 * t + 2 * s + 1];
        acc += 0.5 * double(p.k_b) * (1.0 - (cos_t * c0 + sin_t * s0));
      }
    }
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
      double di[3], u[3];
      const double w0 = p.vtx_w[i];
      for (int k = 0; k < 3; ++k) {
        di[k] = double(p.d[base + k * n_pad + i]);
        u[k] = w0 * di[k];
      }
      for (int q = 0; q < p.valence_max; ++q) {
        const int j = p.vtx_nbr[q * n + i];
        const double w = p.vtx_w[(q + 1) * n + i];
        for (int k = 0; k < 3; ++k) u[k] += w * double(p.d[base + k * n_pad + j]);
      }
      // d^T M~ d / (2 h^2) = 1/2 [inertia_coef m |d|^2 + (beta/h)(k_mem d.L_cot d + k_b |L_cot d|^2 / A_v)]
      const double dd = dot3(di, di), du = dot3(di, u), uu = dot3(u, u);
      acc += 0.5 * (double(p.inertia_coef) * double(p.vtx_mass[i]) * dd +
                    double(p.beta_over_h) * (double(p.k_mem) * du + double(p.k_b) * double(p.vtx_inv_area[i]) * uu));
      for (int k = 0; k < 3; ++k) acc -= di[k] * double(p.b[base + k * n_pad + i]);
    }
    // reduce acc and vol
    double two[2] = {acc, vol};
    for (int r = 0; r < 2; ++r) {
      double v = two[r];
      for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
      __syncthreads();
      if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
      __syncthreads();
      double s = 0.0;
      for (int i = 0; i < int(blockDim.x >> 5); ++i) s += red[i];
      two[r] = s;
    }
    if (threadIdx.x == 0) {
      const double V = two[1] / 6.0, V0 = double(p.V0);
      out_row[cell_id ? cell_id[cell] : cell] = two[0] + 0.5 * double(p.kv_over_V0) * (V - V0) * (V - V0);
    }
    __syncthreads();
  }
  (void)h;
}

// two consecutive table entries with one 8- / 16-byte load (a strided scalar load costs a wavefront per 128 bytes touched)
__device__ __forceinline__ void load_pair(const float *p, double &a, double &b) {
  const float2 v = *reinterpret_cast<const float2 *>(p);
  a = double(v.x);
  b = double(v.y);
}
__device__ __forceinline__ void load_pair(const double *p, double &a, double &b) {
  const double2 v = *reinterpret_cast<const double2 *>(p);
  a = v.x;
  b = v.y;
}

// ---- objective, shared-memory version (line search): the same sum as objective_kernel
// with x_n + d and the UNIT triangle normals of the cell staged once in shared memory in fp64, so a hinge
// costs one rsqrt (1/|e|) instead of three neighbour-normal cross products, two sqrt and a division.
// d itself is staged too (compute type): the damping part's one-ring stencil then gathers from shared memory instead
// of issuing ~20 scattered global loads per vertex.
// Shared memory: 8 (3 n + 3 T) + 3 n sizeof(T) bytes (RBC-642 fp32: 54 KB, RBC-2562: 215 KB); larger meshes keep
// objective_kernel.
template <typename T, int NT>
__global__ void __launch_bounds__(NT)
objective_smem_kernel(const LocalParams<T> p, const int64_t *__restrict__ cell_id, double *__restrict__ out_row,
                      const int *__restrict__ skip) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ double red[2][NT / 32];
  const int n = p.n, n_pad = p.n_pad, nt = p.T_;
  double *sp = reinterpret_cast<double *>(smem_raw);   // [3][n] x_n + d
  double *sn = sp + 3 * n;                              // [T][3] unit normals
  T *sd = reinterpret_cast<T *>(sn + 3 * nt);           // [3][n] d
  if (skip && skip[p.cells] == 0) return;               // line search: skip[cells] = cells still searching
  for (int64_t cell = blockIdx.x; cell < p.cells; cell += gridDim.x) {
    if (skip && skip[cell]) continue;                   // uniform over the CTA
    const size_t base = size_t(cell) * 3 * n_pad;
    for (int k = 0; k < 3; ++k)
      for (int i = threadIdx.x; i < n; i += NT) {
        const T di = p.d[base + k * n_pad + i];
        sd[k * n + i] = di;
        sp[k * n + i] = double(p.x[base + k * n_pad + i]) + ((p.xl ? double(p.xl[base + k * n_pad + i]) : 0.0) + double(di));
      }
    __syncthreads();
    double acc = 0.0, vol = 0.0;
    for (int t = threadIdx.x; t < nt; t += NT) {
      const int4 tv = p.tri[t];
      double x0[3], e1[3], e2[3], N[3];
      for (int k = 0; k < 3; ++k) {
        x0[k] = sp[k * n + tv.x];
        e1[k] = sp[k * n + tv.y] - x0[k];
        e2[k] = sp[k * n + tv.z] - x0[k];
      }
      cross3(e1, e2, N);
      vol += dot3(x0, N);
      double a, b, c, A0;
      load_pair(p.tri_rest + 4 * t, a, b);
      load_pair(p.tri_rest + 4 * t + 2, c, A0);
      const double e11 = dot3(e1, e1), e12 = dot3(e1, e2), e22 = dot3(e2, e2);
      const double C11 = a * a * e11, C12 = a * (b * e11 + c * e12), C22 = b * b * e11 + 2 * b * c * e12 + c * c * e22;
      const double I1 = C11 + C22 - 2.0, I2 = C11 * C22 - C12 * C12 - 1.0;
      acc += A0 * (double(p.B4) * (0.5 * I1 * I1 + I1 - I2) + 0.5 * double(p.C4) * I2 * I2);
      const double rn = rsqrt(dot3(N, N));
      for (int k = 0; k < 3; ++k) sn[3 * t + k] = N[k] * rn;
    }
    __syncthreads();
    for (int t = threadIdx.x; t < nt; t += NT) {
      const int4 tv = p.tri[t];
      const int4 tn = p.tri_nbr[t];
      const int nb[3] = {tn.x, tn.y, tn.z};
      const int vs[3] = {tv.x, tv.y, tv.z};
      const double N[3] = {sn[3 * t], sn[3 * t + 1], sn[3 * t + 2]};
      for (int s = 0; s < 3; ++s) {   // every hinge is seen from both of its triangles: half each
        const double NB[3] = {sn[3 * nb[s]], sn[3 * nb[s] + 1], sn[3 * nb[s] + 2]};
        double e[3], cr[3];
        for (int k = 0; k < 3; ++k) e[k] = sp[k * n + vs[(s + 1) % 3]] - sp[k * n + vs[s]];
        cross3(N, NB, cr);
        const double sin_t = dot3(cr, e) * rsqrt(dot3(e, e)), cos_t = dot3(N, NB);
        double c0, s0;
        load_pair(p.hinge_rest + 6 * t + 2 * s, c0, s0);
        acc += 0.5 * double(p.k_b) * (1.0 - (cos_t * c0 + sin_t * s0));
      }
    }
    for (int i = threadIdx.x; i < n; i += NT) {
      double di[3], u[3];
      const double w0 = p.vtx_w[i];
      for (int k = 0; k < 3; ++k) {
        di[k] = double(sd[k * n + i]);
        u[k] = w0 * di[k];
      }
      for (int q = 0; q < p.valence_max; ++q) {
        const int j = p.vtx_nbr[q * n + i];
        const double w = p.vtx_w[(q + 1) * n + i];
        for (int k = 0; k < 3; ++k) u[k] += w * double(sd[k * n + j]);
      }
      const double dd = dot3(di, di), du = dot3(di, u), uu = dot3(u, u);
      acc += 0.5 * (double(p.inertia_coef) * double(p.vtx_mass[i]) * dd +
                    double(p.beta_over_h) * (double(p.k_mem) * du + double(p.k_b) * double(p.vtx_inv_area[i]) * uu));
      for (int k = 0; k < 3; ++k) acc -= di[k] * double(p.b[base + k * n_pad + i]);
    }
    for (int o = 16; o > 0; o >>= 1) {
      acc += __shfl_xor_sync(0xffffffffu, acc, o);
      vol += __shfl_xor_sync(0xffffffffu, vol, o);
    }
    if ((threadIdx.x & 31) == 0) {
      red[0][threadIdx.x >> 5] = acc;
      red[1][threadIdx.x >> 5] = vol;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
      double sa = 0.0, sv = 0.0;
      for (int i = 0; i < NT / 32; ++i) {
        sa += red[0][i];
        sv += red[1][i];
      }
      const double V = sv / 6.0, V0 = double(p.V0);
      out_row[cell_id ? cell_id[cell] : cell] = sa + 0.5 * double(p.kv_over_V0) * (V - V0) * (V - V0);
    }
    __syncthreads();   // red and the staged cell are reused by the next cell
  }
}

template <typename T>
LocalParams<T> make_params(const TypeDev &td, const BucketView &bv) {
  LocalParams<T> p;
  p.n = td.n; p.T_ = td.T; p.n_pad = td.n_pad; p.valence_max = td.valence_max;
  p.tri = td.tri; p.tri_nbr = td.tri_nbr;
  p.tri_rest = static_cast<const T *>(td.tri_rest);
  p.hinge_rest = static_cast<const T *>(td.hinge_rest);
  p.vtx_corner = td.vtx_corner; p.vtx_nbr = td.vtx_nbr;
  p.vtx_w = static_cast<const T *>(td.vtx_w);
  p.vtx_mass = static_cast<const T *>(td.vtx_mass);
  p.vtx_inv_area = static_cast<const T *>(td.vtx_inv_area);
  p.B4 = T(td.B4); p.C4 = T(td.C4); p.k_b = T(td.k_b); p.kv_over_V0 = T(td.kv_over_V0); p.V0 = T(td.V0);
  p.k_mem = T(td.k_mem); p.beta_over_h = T(td.beta_over_h); p.inertia_coef = T(td.inertia_coef);
  p.x = static_cast<const T *>(bv.field[F_X]);
  p.xl = static_cast<const T *>(bv.field[F_XL]);
  p.d = static_cast<const T *>(bv.field[F_D]);
  p.b = static_cast<const T *>(bv.field[F_B]);
  p.g = static_cast<T *>(bv.field[F_G]);
  p.g_tf32 = bv.g_tf32;
  p.cells = bv.cells;
  p.scratch = nullptr;
  p.scratch_in_smem = 1;
  return p;
}

constexpr size_t kMaxSmem = 200 * 1024;

template <typename T>
size_t smem_full(const TypeDev &td) { return sizeof(T) * (size_t(9) * td.n + size_t(13) * td.T); }
template <typename T>
size_t smem_min(const TypeDev &td) { return sizeof(T) * size_t(9) * td.n; }

template <typename T>
int launch_local_T(const TypeDev &td, const BucketView &bv, void *scratch, int n_sm, cudaStream_t s) {
  LocalParams<T> p = make_params<T>(td, bv);
  size_t smem = smem_full<T>(td);
  if (smem > kMaxSmem) {
    smem = smem_min<T>(td);
    p.scratch_in_smem = 0;
    p.scratch = static_cast<T *>(scratch);
    if (smem > kMaxSmem) {                   // e.g. a 10,242-vertex level-5 mesh: the vertex arrays go to the slab too
      smem = 0;
      p.scratch_in_smem = -1;
    }
  }
  if (!td.cache.generic_attr[sizeof(T) == 8]) {   // per context and type (the attribute is per device)
    if (cudaFuncSetAttribute(local_generic_kernel<T, 256>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(kMaxSmem)) != cudaSuccess ||
        cudaFuncSetAttribute(local_generic_kernel<T, 512>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(kMaxSmem)) != cudaSuccess)
      return -1;
    td.cache.generic_attr[sizeof(T) == 8] = true;
  }
  const int per_sm = smem * 2 + 4096 <= 227 * 1024 ? 2 : 1;
  int64_t grid = int64_t(n_sm) * per_sm;
  if (grid > bv.cells) grid = bv.cells;
  // one CTA per SM (fp64, large meshes): 512 threads with up to 128 registers each hide the FP64 latencies
  if (per_sm == 1)
    local_generic_kernel<T, 512><<<unsigned(grid), 512, smem, s>>>(p);
  else
    local_generic_kernel<T, 256><<<unsigned(grid), 256, smem, s>>>(p);
  return 1;
}

}  // namespace

size_t local_generic_scratch_bytes(const TypeDev &td, int precision, int n_sm) {
  const size_t es = precision == NPFEM_F32 ? 4 : 8;
  const size_t full = es * (size_t(9) * td.n + size_t(13) * td.T);
  if (full <= kMaxSmem) return 0;
  const size_t per_cta = es * size_t(9) * td.n <= kMaxSmem ? es * size_t(13) * td.T : full;
  return per_cta * size_t(n_sm) * 2;
}

int launch_local_generic(const TypeDev &td, const BucketView &bv, void *scratch, int precision, int n_sm,
                         cudaStream_t s) {
  if (bv.cells == 0) return 0;
  return precision == NPFEM_F32 ? launch_local_T<float>(td, bv, scratch, n_sm, s)
                                : launch_local_T<double>(td, bv, scratch, n_sm, s);
}

template <typename T>
int launch_objective_T(const TypeDev &td, const BucketView &bv, const int64_t *cell_id_dev, double *objective_row,
                       const int *skip_dev, int n_sm, cudaStream_t s) {
  const LocalParams<T> p = make_params<T>(td, bv);
  const size_t smem = sizeof(double) * (size_t(3) * td.n + size_t(3) * td.T) + sizeof(T) * size_t(3) * td.n;
  if (smem <= 74 * 1024) {                    // 4 (fp32 RBC-642: 54 KB each) or 3 (fp64: 62 KB) CTAs of 256 threads per SM
    if (!td.cache.objective_attr) cudaFuncSetAttribute(objective_smem_kernel<T, 256>, cudaFuncAttributeMaxDynamicSharedMemorySize, 74 * 1024);
    td.cache.objective_attr = true;
    const int64_t cap = int64_t(n_sm) * (smem <= 56 * 1024 ? 4 : 3) * 4;
    objective_smem_kernel<T, 256><<<unsigned(bv.cells < cap ? bv.cells : cap), 256, smem, s>>>(p, cell_id_dev, objective_row, skip_dev);
  } else if (smem <= kMaxSmem) {              // one CTA of 1024 threads per SM (RBC-2562: 184 KB)
    if (!td.cache.objective_attr) cudaFuncSetAttribute(objective_smem_kernel<T, 1024>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(kMaxSmem));
    td.cache.objective_attr = true;
    const int64_t cap = int64_t(n_sm) * 4;
    objective_smem_kernel<T, 1024><<<unsigned(bv.cells < cap ? bv.cells : cap), 1024, smem, s>>>(p, cell_id_dev, objective_row, skip_dev);
  } else {
    objective_kernel<T><<<unsigned(bv.cells < 148 * 8 ? bv.cells : 148 * 8), 256, 0, s>>>(p, cell_id_dev, objective_row, skip_dev, td.h);
  }
  return 1;
}

int launch_objective(const TypeDev &td, const BucketView &bv, const int64_t *cell_id_dev, double *objective_row,
                     const int *skip_dev, int precision, int n_sm, cudaStream_t s) {
  if (bv.cells == 0) return 0;
  return precision == NPFEM_F32 ? launch_objective_T<float>(td, bv, cell_id_dev, objective_row, skip_dev, n_sm, s)
                                : launch_objective_T<double>(td, bv, cell_id_dev, objective_row, skip_dev, n_sm, s);
}

}  // namespace npfem
