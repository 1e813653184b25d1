// Local step (row a2), fp32, for cell types too large for the scheduled kernel (local_sched.cu keeps a
// type's topology in registers: <= 1,362 triangles), e.g. BASELINE config 5's RBC-2562 (5,120 triangles).
// Same arithmetic and the same reduced gradient as the other fp32 fast kernels,
//   r = (1 - gamma) m^ d - b + grad E(x_n + d)   (readings R5-R9; local_smem.cu),
// so the global step runs with d_scale = 1 - gamma.
//
// One persistent CTA of 1024 threads per SM, one cell at a time.  Positions (float4) and unit normals
// (float4) of the WHOLE cell live in shared memory; corner forces do not fit next to them, so phase B
// runs in NCH chunks of triangles: each chunk writes its corner forces to a shared buffer, then every
// thread adds the corners of ITS vertices that fall into the chunk to register accumulators (fixed
// order: deterministic, no atomics).  The per-type tables (packed 16-bit connectivity, Dm^-1, rest
// hinge angles, vertex incidence) stream from L2 (they are the same for every cell).
// The generic kernel it replaces on this path kept normals and corner forces in a GLOBAL scratch:
// 4.1 ms per launch at 10,000 RBC-2562 (4.5 % of HBM peak).
#include "internal.h"

namespace npfem {
namespace {

constexpr int THREADS = 1024;
constexpr int VPT = 4;        // vertices per thread (n <= 4096)

struct BigParams {
  int n, T, n_pad, tc;        // tc: triangles per chunk
  const uint4 *tri_pack;      // [T]  v0|v1<<16, v2|n0<<16, n1|n2<<16, 0
  const float4 *tri_rest;     // [T]  a b c A0
  const float2 *hinge_rest;   // [T][3] (cos, sin) theta0
  const uint4 *vtx_pack;      // [n]  8 x u16 corner ids, 3T = none
  const float *vtx_coef;      // [n]  (1 - gamma)(1 + h alpha) m_v / h^2
  float B4, C4, k_b;
  double kv_over_V0, V0;
  const float *x, *xl, *d, *b;   // [cells][3][n_pad]; positions are the two-float sum x + xl (internal.h F_XL)
  float *g;
  int g_tf32;
  int64_t cells;
};

__device__ __forceinline__ float rsqrt_fast(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

__global__ void __launch_bounds__(THREADS, 1) local_big_kernel(const BigParams p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ double red[32];
  const int n = p.n, nt = p.T, n_pad = p.n_pad, tc = p.tc;
  float4 *sx = reinterpret_cast<float4 *>(smem_raw);     // [n]  x_n + d
  float4 *sN = sx + n;                                   // [T]  unit normal, 1/|N|
  float4 *sC = sN + nt;                                  // [3 tc] corner forces of the current chunk
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

  for (int64_t cell = blockIdx.x; cell < p.cells; cell += gridDim.x) {
    const size_t base = size_t(cell) * 3 * n_pad;
    const float *xg = p.x + base, *lg = p.xl + base, *dg = p.d + base, *bg = p.b + base;
    {   // pull the NEXT cell's x, d, b towards L2 while this one is computed (one 128-byte line per thread)
      const int64_t nxt = cell + gridDim.x;
      const int lines = (3 * n_pad * 4 + 127) / 128;
      if (nxt < p.cells)
        for (int l = tid; l < 4 * lines; l += THREADS) {
          const float *f = (l < lines ? p.x : (l < 2 * lines ? p.d : (l < 3 * lines ? p.b : p.xl))) + size_t(nxt) * 3 * n_pad;
          asm volatile("prefetch.global.L2 [%0];" ::"l"(reinterpret_cast<const char *>(f) + size_t(l % lines) * 128));
        }
    }
    // ---- phase 0 ----------------------------------------------------------------------------
    for (int i = tid; i < n; i += THREADS)
      sx[i] = make_float4(xg[i] + (lg[i] + dg[i]), xg[n_pad + i] + (lg[n_pad + i] + dg[n_pad + i]),
                          xg[2 * n_pad + i] + (lg[2 * n_pad + i] + dg[2 * n_pad + i]), 0.f);   // two-float x_n (F_XL)
    __syncthreads();
    // ---- phase A: unit normals, volume --------------------------------------------------------
    float vol = 0.f;
    for (int t = tid; t < nt; t += THREADS) {
      const uint4 pk = __ldg(p.tri_pack + t);
      const float4 X0 = sx[pk.x & 0xffffu], X1 = sx[pk.x >> 16], X2 = sx[pk.y & 0xffffu];
      const float e1x = X1.x - X0.x, e1y = X1.y - X0.y, e1z = X1.z - X0.z;
      const float e2x = X2.x - X0.x, e2y = X2.y - X0.y, e2z = X2.z - X0.z;
      const float Nx = e1y * e2z - e1z * e2y, Ny = e1z * e2x - e1x * e2z, Nz = e1x * e2y - e1y * e2x;
      const float inv = rsqrt_fast(Nx * Nx + Ny * Ny + Nz * Nz);
      sN[t] = make_float4(Nx * inv, Ny * inv, Nz * inv, inv);
      vol += X0.x * Nx + X0.y * Ny + X0.z * Nz;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) vol += __shfl_xor_sync(0xffffffffu, vol, o);
    if (lane == 0) red[warp] = double(vol);
    __syncthreads();
    float vc;
    {
      double v = red[lane];                               // 32 warps
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
      vc = float(p.kv_over_V0 * (v * (1.0 / 6.0) - p.V0) * (1.0 / 6.0));   // k_v (V - V0)/V0 / 6
    }
    // ---- phases B + C, chunk by chunk ---------------------------------------------------------
    float acc[VPT][3];
#pragma unroll
    for (int r = 0; r < VPT; ++r) acc[r][0] = acc[r][1] = acc[r][2] = 0.f;
    for (int t0 = 0; t0 < nt; t0 += tc) {
      const int t1 = min(t0 + tc, nt);
      // the per-type tables come from L2: the next triangle's entries are requested before this one is
      // worked on (one L2 latency per chunk instead of one per triangle)
      int t = t0 + tid;
      uint4 pk_n = make_uint4(0, 0, 0, 0);
      float4 rest_n = make_float4(0.f, 0.f, 0.f, 0.f);
      float2 h_n[3] = {};
      if (t < t1) {
        pk_n = __ldg(p.tri_pack + t);
        rest_n = __ldg(p.tri_rest + t);
#pragma unroll
        for (int sd = 0; sd < 3; ++sd) h_n[sd] = __ldg(p.hinge_rest + 3 * t + sd);
      }
      for (; t < t1; t += THREADS) {
        const uint4 pk = pk_n;
        const float4 rest = rest_n;
        const float2 hh[3] = {h_n[0], h_n[1], h_n[2]};
        if (t + THREADS < t1) {
          pk_n = __ldg(p.tri_pack + t + THREADS);
          rest_n = __ldg(p.tri_rest + t + THREADS);
#pragma unroll
          for (int sd = 0; sd < 3; ++sd) h_n[sd] = __ldg(p.hinge_rest + 3 * (t + THREADS) + sd);
        }
        const float4 X0 = sx[pk.x & 0xffffu], X1 = sx[pk.x >> 16], X2 = sx[pk.y & 0xffffu];
        const float4 NA = sN[t];
        const float a = rest.x, b = rest.y, c = rest.z, A0 = rest.w;
        const float e1[3] = {X1.x - X0.x, X1.y - X0.y, X1.z - X0.z};
        const float e2[3] = {X2.x - X0.x, X2.y - X0.y, X2.z - X0.z};
        const float e11 = e1[0] * e1[0] + e1[1] * e1[1] + e1[2] * e1[2];
        const float e12 = e1[0] * e2[0] + e1[1] * e2[1] + e1[2] * e2[2];
        const float e22 = e2[0] * e2[0] + e2[1] * e2[1] + e2[2] * e2[2];
        // membrane (Skalak): Q = 2 A0 (W1 R + W2 det^2 adj G), R = Dm^-1 Dm^-T, det = a c
        const float R11 = a * a + b * b, R12 = b * c, R22 = c * c, J = (a * c) * (a * c);
        const float nn = 1.f / (NA.w * NA.w);
        const float I1p1 = R11 * e11 + 2.f * R12 * e12 + R22 * e22 - 1.f, I2 = J * nn - 1.f;
        const float W1 = 2.f * A0 * p.B4 * I1p1, W2 = 2.f * A0 * J * (p.C4 * I2 - p.B4);
        const float q11 = W1 * R11 + W2 * e22, q22 = W1 * R22 + W2 * e11, q12 = W1 * R12 - W2 * e12;
        // hinges seen from this triangle: side s from corner s to s+1
        float w0 = 0.f, w1 = 0.f, w2 = 0.f;
        const uint32_t nbr[3] = {pk.y >> 16, pk.z & 0xffffu, pk.z >> 16};
        const float len2[3] = {e11, e11 - 2.f * e12 + e22, e22};
        const float djk[3] = {e11 - e12, e22 - e12, e12};
#pragma unroll
        for (int s = 0; s < 3; ++s) {
          const float4 NB = sN[nbr[s]];
          const float2 h0 = hh[s];
          const float ex = s == 0 ? e1[0] : (s == 1 ? e2[0] - e1[0] : -e2[0]);
          const float ey = s == 0 ? e1[1] : (s == 1 ? e2[1] - e1[1] : -e2[1]);
          const float ez = s == 0 ? e1[2] : (s == 1 ? e2[2] - e1[2] : -e2[2]);
          const float crx = NA.y * NB.z - NA.z * NB.y, cry = NA.z * NB.x - NA.x * NB.z, crz = NA.x * NB.y - NA.y * NB.x;
          const float ie = rsqrt_fast(len2[s]);
          const float S = crx * ex + cry * ey + crz * ez, cs = NA.x * NB.x + NA.y * NB.y + NA.z * NB.z;
          const float q = p.k_b * ie * (S * ie * h0.x - cs * h0.y);          // dE/dtheta / |e|
          const float ci = djk[s] * q, cj = (len2[s] - djk[s]) * q, ck = -len2[s] * q;
          if (s == 0) { w0 += ci; w1 += cj; w2 += ck; }
          if (s == 1) { w1 += ci; w2 += cj; w0 += ck; }
          if (s == 2) { w2 += ci; w0 += cj; w1 += ck; }
        }
        const float vn = vc * (nn * NA.w);                                   // vc |N|
        const float u0 = NA.w * w0 + vn, u1 = NA.w * w1 + vn, u2 = NA.w * w2 + vn, us = u0 + u1 + u2;
        const float nA[3] = {NA.x, NA.y, NA.z};
        float c0[3], c1[3], c2[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
          c1[k] = u1 * nA[k] + q11 * e1[k] + q12 * e2[k];
          c2[k] = u2 * nA[k] + q12 * e1[k] + q22 * e2[k];
          c0[k] = us * nA[k] - c1[k] - c2[k];
        }
        const int o = 3 * (t - t0);
        sC[o] = make_float4(c0[0], c0[1], c0[2], 0.f);
        sC[o + 1] = make_float4(c1[0], c1[1], c1[2], 0.f);
        sC[o + 2] = make_float4(c2[0], c2[1], c2[2], 0.f);
      }
      __syncthreads();                                    // this chunk's corner forces complete
      const uint32_t lo = 3u * uint32_t(t0), hi = 3u * uint32_t(t1);
#pragma unroll
      for (int r = 0; r < VPT; ++r) {
        const int i = tid + r * THREADS;
        if (i < n) {
          const uint4 pk = __ldg(p.vtx_pack + i);
          const uint32_t w[4] = {pk.x, pk.y, pk.z, pk.w};
#pragma unroll
          for (int q = 0; q < 8; ++q) {
            const uint32_t cid = (q & 1) ? (w[q >> 1] >> 16) : (w[q >> 1] & 0xffffu);
            if (cid >= lo && cid < hi) {
              const float4 f = sC[cid - lo];
              acc[r][0] += f.x; acc[r][1] += f.y; acc[r][2] += f.z;
            }
          }
        }
      }
      __syncthreads();                                    // sC can be overwritten by the next chunk
    }
    // ---- write the reduced gradient -------------------------------------------------------------
#pragma unroll
    for (int r = 0; r < VPT; ++r) {
      const int i = tid + r * THREADS;
      if (i < n) {
        const float coef = __ldg(p.vtx_coef + i);
        const float g0 = coef * dg[i] - bg[i] + acc[r][0], g1 = coef * dg[n_pad + i] - bg[n_pad + i] + acc[r][1],
                    g2 = coef * dg[2 * n_pad + i] - bg[2 * n_pad + i] + acc[r][2];
        p.g[base + i] = p.g_tf32 ? tf32_rn(g0) : g0;
        p.g[base + n_pad + i] = p.g_tf32 ? tf32_rn(g1) : g1;
        p.g[base + 2 * n_pad + i] = p.g_tf32 ? tf32_rn(g2) : g2;
      }
    }
    // the next cell's phase 0 writes sx: every thread is past its last read of sx (phase B) here
  }
}

int chunk_triangles(int n, int T) {     // largest chunk whose corner buffer fits next to sx and sN
  const size_t fixed = size_t(n) * 16 + size_t(T) * 16;
  const size_t budget = 224 * 1024;
  if (fixed + 3 * 16 * 256 > budget) return 0;
  size_t tc = (budget - fixed) / 48;
  if (tc > size_t(T)) tc = size_t(T);
  const int chunks = int((T + tc - 1) / tc);
  return (T + chunks - 1) / chunks;     // equal chunks
}

}  // namespace

bool local_big_supported(const TypeDev &td) {
  return td.tri_pack != nullptr && td.valence_max <= 8 && td.n <= THREADS * VPT && chunk_triangles(td.n, td.T) > 0;
}

int launch_local_big(const TypeDev &td, const BucketView &bv, int n_sm, cudaStream_t s) {
  if (bv.cells == 0) return 0;
  if (!local_big_supported(td)) return -1;
  BigParams p;
  p.n = td.n; p.T = td.T; p.n_pad = td.n_pad; p.tc = chunk_triangles(td.n, td.T);
  p.tri_pack = static_cast<const uint4 *>(td.tri_pack);
  p.tri_rest = static_cast<const float4 *>(td.tri_rest);
  p.hinge_rest = static_cast<const float2 *>(td.hinge_rest);
  p.vtx_pack = static_cast<const uint4 *>(td.vtx_pack);
  p.vtx_coef = static_cast<const float *>(td.vtx_coef);
  p.B4 = float(td.B4); p.C4 = float(td.C4); p.k_b = float(td.k_b);
  p.kv_over_V0 = td.kv_over_V0; p.V0 = td.V0;
  p.x = static_cast<const float *>(bv.field[F_X]);
  p.xl = static_cast<const float *>(bv.field[F_XL]);
  p.d = static_cast<const float *>(bv.field[F_D]);
  p.b = static_cast<const float *>(bv.field[F_B]);
  p.g = static_cast<float *>(bv.field[F_G]);
  p.g_tf32 = bv.g_tf32;
  p.cells = bv.cells;
  const size_t smem = size_t(td.n) * 16 + size_t(td.T) * 16 + size_t(3) * p.tc * 16;
  if (!td.cache.big_attr) {   // per context (the attribute is per device): always the architectural maximum
    if (opt_in_max_dynamic_smem(local_big_kernel) != cudaSuccess) return -1;
    td.cache.big_attr = true;
  }
  const int64_t grid = bv.cells < n_sm ? bv.cells : n_sm;
  local_big_kernel<<<unsigned(grid), THREADS, smem, s>>>(p);
  return 1;
}

}  // namespace npfem
