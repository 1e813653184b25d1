// Local step (row a2), fp32 fast path for cell types whose topology + one cell fit in shared memory
// (RBC-642, PLT-162).  Persistent CTAs: the constant per-TYPE tables (connectivity as packed 16-bit
// indices, Dm^-1, rest areas, rest hinge angles, vertex incidence lists) are loaded into shared memory
// ONCE per launch and reused for every cell the CTA processes; the per-cell state streams in through
// 1-D TMA bulk copies (cp.async.bulk + mbarrier) that are issued one cell ahead.
//
// It writes the REDUCED gradient  r = (1 - gamma) m^ d - b + grad E(x_n + d),  m^ = (1 + h alpha) M / h^2,
// gamma = (beta/h)/(1 + beta/h), for which Eq. (4) reads exactly
//     d <- (1 - gamma) d - H~^-1 r
// because H~ = m^ + (1 + beta/h) L and M~/h^2 = m^ + (beta/h) L  =>  H~^-1 (beta/h) L d =
// gamma (d - H~^-1 m^ d).  The Rayleigh stencil (two one-ring passes of L_cot per iteration) thus
// disappears from the hot loop; the global-step epilogue applies the (1 - gamma) factor.
//
// Phases per cell (3 block barriers):
//   0  staged x_n, d, b -> sx[v] = (x_n + d, 0) as float4;  d_v, b_v stay in registers     | barrier
//      (thread 0 then launches the bulk copies of the NEXT cell into the staging buffer)
//   A  per triangle: N_t = e1 x e2, |N_t|^2 -> sN[t] (float4); volume partial                | barrier
//   B  per triangle: Skalak gradient + 3 hinge sides + volume term -> 3 corner forces (float4)| barrier
//   C  per vertex: gather <= 8 corner slots (fixed order, no atomics), r = coef d - b + sum -> global
#include "internal.h"

namespace npfem {
namespace {

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return uint32_t(__cvta_generic_to_shared(p)); }

struct SmemLocalParams {
  int n, T, n_pad;
  int valence_max;
  const uint4 *tri_pack;     // [T]  v0|v1<<16, v2|n0<<16, n1|n2<<16, 0
  const float4 *tri_rest;    // [T]  a b c A0
  const float2 *hinge_rest;  // [T][3] (cos, sin) theta0
  const uint4 *vtx_pack;     // [n]  8 x u16 corner ids, 0xFFFF = none
  const float *vtx_coef;     // [n]  (1 - gamma) (1 + h alpha) m_v / h^2
  float B4, C4, k_b, kv_over_V0, V0;
  const float *x, *xl, *d, *b;   // [cells][3][n_pad]; positions are the two-float sum x + xl (internal.h F_XL)
  float *g;
  int g_tf32;
  int64_t cells;
};

template <int MAXV_SLOTS>
__global__ void __launch_bounds__(768, 1)
local_smem_kernel(const SmemLocalParams p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int n = p.n, nt = p.T, n_pad = p.n_pad;
  // ---- carve shared memory ----------------------------------------------------------------
  uint4 *s_tri = reinterpret_cast<uint4 *>(smem_raw);
  float4 *s_rest = reinterpret_cast<float4 *>(s_tri + nt);
  float2 *s_hinge = reinterpret_cast<float2 *>(s_rest + nt);
  uint4 *s_vtx = reinterpret_cast<uint4 *>(s_hinge + 3 * nt + (nt & 1));
  float4 *sx = reinterpret_cast<float4 *>(s_vtx + n);
  float4 *sN = sx + n;
  float4 *sC = sN + nt;                                  // [3T + 1], last slot = zero (absent corner)
  float *stage = reinterpret_cast<float *>(sC + 3 * nt + 1);   // [3 fields][3][n_pad]
  float *s_coef = stage + 9 * n_pad;
  double *red = reinterpret_cast<double *>(s_coef + ((n + 3) & ~3));
  uint64_t *mbar = reinterpret_cast<uint64_t *>(red + 32);

  const int tid = threadIdx.x, nthreads = blockDim.x, warp = tid >> 5, lane = tid & 31;
  const uint32_t field_bytes = uint32_t(3 * n_pad) * 4u;

  auto prefetch = [&](int64_t cell) {     // one thread: arm the barrier and start 3 bulk copies
    const size_t base = size_t(cell) * 3 * n_pad;
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(mbar)), "r"(3 * field_bytes)
                 : "memory");
    const float *src[3] = {p.x + base, p.d + base, p.b + base};
#pragma unroll
    for (int f = 0; f < 3; ++f)
      asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                   ::"r"(smem_u32(stage + f * 3 * n_pad)), "l"(src[f]), "r"(field_bytes), "r"(smem_u32(mbar))
                   : "memory");
  };

  if (tid == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(mbar)));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (tid == 0 && int64_t(blockIdx.x) < p.cells) prefetch(blockIdx.x);
  // ---- per-type tables: once per launch -----------------------------------------------------
  for (int t = tid; t < nt; t += nthreads) {
    s_tri[t] = p.tri_pack[t];
    s_rest[t] = p.tri_rest[t];
    s_hinge[3 * t] = p.hinge_rest[3 * t];
    s_hinge[3 * t + 1] = p.hinge_rest[3 * t + 1];
    s_hinge[3 * t + 2] = p.hinge_rest[3 * t + 2];
  }
  for (int i = tid; i < n; i += nthreads) {
    s_vtx[i] = p.vtx_pack[i];
    s_coef[i] = p.vtx_coef[i];
  }
  if (tid == 0) sC[3 * nt] = make_float4(0.f, 0.f, 0.f, 0.f);
  __syncthreads();

  uint32_t parity = 0;
  for (int64_t cell = blockIdx.x; cell < p.cells; cell += gridDim.x) {
    const size_t base = size_t(cell) * 3 * n_pad;
    // ---- phase 0 ----------------------------------------------------------------------------
    {
      uint32_t done;
      do {
        asm volatile(
            "{\n.reg .pred q;\nmbarrier.try_wait.parity.shared::cta.b64 q, [%1], %2;\nselp.u32 %0, 1, 0, q;\n}\n"
            : "=r"(done) : "r"(smem_u32(mbar)), "r"(parity) : "memory");
      } while (!done);
      parity ^= 1;
    }
    float dv[2][3], bv[2][3];
#pragma unroll
    for (int r = 0; r < 2; ++r) {
      const int i = tid + r * nthreads;
      if (i < n) {
        float xs[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
          dv[r][k] = stage[(3 + k) * n_pad + i];
          bv[r][k] = stage[(6 + k) * n_pad + i];
          xs[k] = stage[k * n_pad + i] + (__ldg(p.xl + base + k * n_pad + i) + dv[r][k]);
        }
        sx[i] = make_float4(xs[0], xs[1], xs[2], 0.f);
      }
    }
    __syncthreads();                                           // barrier 1: sx complete, staging consumed
    if (tid == 0 && cell + gridDim.x < p.cells) prefetch(cell + gridDim.x);
    // ---- phase A ----------------------------------------------------------------------------
    float vol = 0.f;
    for (int t = tid; t < nt; t += nthreads) {
      const uint4 pk = s_tri[t];
      const float4 X0 = sx[pk.x & 0xffffu], X1 = sx[pk.x >> 16], X2 = sx[pk.y & 0xffffu];
      const float e1x = X1.x - X0.x, e1y = X1.y - X0.y, e1z = X1.z - X0.z;
      const float e2x = X2.x - X0.x, e2y = X2.y - X0.y, e2z = X2.z - X0.z;
      const float Nx = e1y * e2z - e1z * e2y, Ny = e1z * e2x - e1x * e2z, Nz = e1x * e2y - e1y * e2x;
      sN[t] = make_float4(Nx, Ny, Nz, Nx * Nx + Ny * Ny + Nz * Nz);
      vol += X0.x * Nx + X0.y * Ny + X0.z * Nz;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) vol += __shfl_xor_sync(0xffffffffu, vol, o);
    if (lane == 0) red[warp] = double(vol);
    __syncthreads();                                           // barrier 2: sN complete, partial volumes posted
    {
      double v = lane < (nthreads >> 5) ? red[lane] : 0.0;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
      vol = float(double(p.kv_over_V0) * (v / 6.0 - double(p.V0)) / 6.0);   // k_v (V - V0)/V0 / 6
    }
    const float vol_coef = vol;
    // ---- phase B ----------------------------------------------------------------------------
    for (int t = tid; t < nt; t += nthreads) {
      const uint4 pk = s_tri[t];
      const float4 rest = s_rest[t];
      const float4 X0 = sx[pk.x & 0xffffu], X1 = sx[pk.x >> 16], X2 = sx[pk.y & 0xffffu];
      const float4 NA = sN[t];
      const float a = rest.x, b = rest.y, c = rest.z, A0 = rest.w;
      const float e1[3] = {X1.x - X0.x, X1.y - X0.y, X1.z - X0.z};
      const float e2[3] = {X2.x - X0.x, X2.y - X0.y, X2.z - X0.z};
      const float e11 = e1[0] * e1[0] + e1[1] * e1[1] + e1[2] * e1[2];
      const float e12 = e1[0] * e2[0] + e1[1] * e2[1] + e1[2] * e2[2];
      const float e22 = e2[0] * e2[0] + e2[1] * e2[1] + e2[2] * e2[2];
      // membrane (Skalak): F = [a e1, b e1 + c e2], C = F^T F
      const float C11 = a * a * e11;
      const float C12 = a * (b * e11 + c * e12);
      const float C22 = b * b * e11 + 2.f * b * c * e12 + c * c * e22;
      const float I1 = C11 + C22 - 2.f;
      const float I2 = C11 * C22 - C12 * C12 - 1.f;
      const float W1 = p.B4 * (I1 + 1.f);
      const float W2 = p.C4 * I2 - p.B4;
      const float S11 = 2.f * (W1 + W2 * C22), S12 = -2.f * W2 * C12, S22 = 2.f * (W1 + W2 * C11);
      const float p11 = S11 * a + S12 * b, p12 = S12 * c, p21 = S12 * a + S22 * b, p22 = S22 * c;
      const float al1 = A0 * (a * p11 + b * p21), al2 = A0 * (a * p12 + b * p22);
      const float be1 = A0 * c * p21, be2 = A0 * c * p22;
      // hinges seen from this triangle: edge s from corner s to s+1, opposite corner s+2
      float w0 = vol_coef, w1 = vol_coef, w2 = vol_coef;
      const float inv_nnA = __frcp_rn(NA.w);
      const uint32_t nbr[3] = {pk.y >> 16, pk.z & 0xffffu, pk.z >> 16};
      const float len2[3] = {e11, e11 - 2.f * e12 + e22, e22};
      const float djk[3] = {e11 - e12, e22 - e12, e12};
#pragma unroll
      for (int s = 0; s < 3; ++s) {
        const float4 NB = sN[nbr[s]];
        const float2 h0 = s_hinge[3 * t + s];
        const float ex = s == 0 ? e1[0] : (s == 1 ? e2[0] - e1[0] : -e2[0]);
        const float ey = s == 0 ? e1[1] : (s == 1 ? e2[1] - e1[1] : -e2[1]);
        const float ez = s == 0 ? e1[2] : (s == 1 ? e2[2] - e1[2] : -e2[2]);
        const float crx = NA.y * NB.z - NA.z * NB.y, cry = NA.z * NB.x - NA.x * NB.z, crz = NA.x * NB.y - NA.y * NB.x;
        const float inv_e = rsqrtf(len2[s]);
        const float inv_nn = rsqrtf(NA.w * NB.w);
        const float sin_t = (crx * ex + cry * ey + crz * ez) * inv_e * inv_nn;
        const float cos_t = (NA.x * NB.x + NA.y * NB.y + NA.z * NB.z) * inv_nn;
        const float dE = p.k_b * (sin_t * h0.x - cos_t * h0.y);       // k_b sin(theta - theta0)
        const float common = dE * inv_e * inv_nnA;                    // dE / (|e| |N_A|^2)
        const float ci = djk[s] * common, cj = (len2[s] - djk[s]) * common, ck = -len2[s] * common;
        if (s == 0) { w0 += ci; w1 += cj; w2 += ck; }
        if (s == 1) { w1 += ci; w2 += cj; w0 += ck; }
        if (s == 2) { w2 += ci; w0 += cj; w1 += ck; }
      }
      float c0[3], c1[3], c2[3];
      const float Nv[3] = {NA.x, NA.y, NA.z};
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        const float g1 = al1 * e1[k] + al2 * e2[k];
        const float g2 = be1 * e1[k] + be2 * e2[k];
        c0[k] = w0 * Nv[k] - (g1 + g2);
        c1[k] = w1 * Nv[k] + g1;
        c2[k] = w2 * Nv[k] + g2;
      }
      sC[3 * t + 0] = make_float4(c0[0], c0[1], c0[2], 0.f);
      sC[3 * t + 1] = make_float4(c1[0], c1[1], c1[2], 0.f);
      sC[3 * t + 2] = make_float4(c2[0], c2[1], c2[2], 0.f);
    }
    __syncthreads();                                           // barrier 3: corner forces complete
    // ---- phase C ----------------------------------------------------------------------------
#pragma unroll
    for (int r = 0; r < 2; ++r) {
      const int i = tid + r * nthreads;
      if (i < n) {
        const uint4 pk = s_vtx[i];
        const uint32_t w[4] = {pk.x, pk.y, pk.z, pk.w};
        float ax = 0.f, ay = 0.f, az = 0.f;
#pragma unroll
        for (int q = 0; q < MAXV_SLOTS; ++q) {
          const uint32_t cid = (q & 1) ? (w[q >> 1] >> 16) : (w[q >> 1] & 0xffffu);
          const float4 f = sC[cid];
          ax += f.x;
          ay += f.y;
          az += f.z;
        }
        const float coef = s_coef[i];
        const float g0 = coef * dv[r][0] - bv[r][0] + ax, g1 = coef * dv[r][1] - bv[r][1] + ay, g2 = coef * dv[r][2] - bv[r][2] + az;
        p.g[base + i] = p.g_tf32 ? tf32_rn(g0) : g0;
        p.g[base + n_pad + i] = p.g_tf32 ? tf32_rn(g1) : g1;
        p.g[base + 2 * n_pad + i] = p.g_tf32 ? tf32_rn(g2) : g2;
      }
    }
    // no barrier here: the next cell's phase 0 only writes sx (last read before barrier 3) and the
    // staging buffer (consumed before barrier 1); sN / sC are rewritten after barriers 1 / 2
  }
}

}  // namespace

size_t local_smem_bytes(int n, int T, int n_pad) {
  size_t b = 0;
  b += size_t(T) * 16;                 // s_tri
  b += size_t(T) * 16;                 // s_rest
  b += (size_t(3) * T + (T & 1)) * 8;  // s_hinge
  b += size_t(n) * 16;                 // s_vtx
  b += size_t(n) * 16;                 // sx
  b += size_t(T) * 16;                 // sN
  b += (size_t(3) * T + 1) * 16;       // sC
  b += size_t(9) * n_pad * 4;          // stage
  b += size_t((n + 3) & ~3) * 4;       // s_coef
  b += 32 * 8 + 16;                    // red, mbar
  return b;
}

bool local_smem_supported(const TypeDev &td) {
  return td.valence_max <= 8 && td.n <= 65534 && 3 * td.T + 1 <= 65535 &&
         local_smem_bytes(td.n, td.T, td.n_pad) <= 220 * 1024 && td.tri_pack != nullptr;
}

int launch_local_smem(const TypeDev &td, const BucketView &bv, int n_sm, cudaStream_t s) {
  if (bv.cells == 0) return 0;
  if (!local_smem_supported(td)) return -1;
  SmemLocalParams p;
  p.n = td.n; p.T = td.T; p.n_pad = td.n_pad; p.valence_max = td.valence_max;
  p.tri_pack = static_cast<const uint4 *>(td.tri_pack);
  p.tri_rest = static_cast<const float4 *>(td.tri_rest);
  p.hinge_rest = static_cast<const float2 *>(td.hinge_rest);
  p.vtx_pack = static_cast<const uint4 *>(td.vtx_pack);
  p.vtx_coef = static_cast<const float *>(td.vtx_coef);
  p.B4 = float(td.B4); p.C4 = float(td.C4); p.k_b = float(td.k_b); p.kv_over_V0 = float(td.kv_over_V0);
  p.V0 = float(td.V0);
  p.x = static_cast<const float *>(bv.field[F_X]);
  p.xl = static_cast<const float *>(bv.field[F_XL]);
  p.d = static_cast<const float *>(bv.field[F_D]);
  p.b = static_cast<const float *>(bv.field[F_B]);
  p.g = static_cast<float *>(bv.field[F_G]);
  p.g_tf32 = bv.g_tf32;
  p.cells = bv.cells;
  const size_t smem = local_smem_bytes(td.n, td.T, td.n_pad);
  // threads: two triangles per thread for big meshes, one for small ones; vertices need <= 2 rounds
  int threads = (td.T >= 640 ? (td.T + 1) / 2 : td.T);
  threads = (threads + 31) / 32 * 32;
  if (threads > 768) threads = 768;
  if (threads * 2 < td.n) return -1;
  int per_sm = int((227 * 1024) / (smem + 1024));
  if (per_sm < 1) return -1;
  if (per_sm * threads > 2048) per_sm = 2048 / threads;
  if (per_sm > 8) per_sm = 8;
  auto kernel = td.valence_max <= 6 ? local_smem_kernel<6> : local_smem_kernel<8>;
  if (!td.cache.smem_attr) {   // per context and type (the attribute is per device)
    if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024) != cudaSuccess) return -1;
    td.cache.smem_attr = true;
  }
  int64_t grid = int64_t(n_sm) * per_sm;
  if (grid > bv.cells) grid = bv.cells;
  kernel<<<unsigned(grid), threads, smem, s>>>(p);
  return 1;
}

}  // namespace npfem
