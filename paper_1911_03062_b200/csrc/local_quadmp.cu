// Local step (row a2), fp32, MULTI-PASS quad path for meshes too large for one pass of the quad kernel (1,282 ... 5,120
// triangles: RBC-2562 of BASELINE configs[4] has 2,560 quads): the arithmetic of local_quad.cu - one thread per pair of
// adjacent triangles T0 = (p, q, r), T1 = (p, s, q), same reduced gradient r = (1 - gamma) m^ d - b + grad E(x_n + d)
// (Eqs. (3)-(4), readings R5-R9) - with the quads of a cell taken in up to 4 PASSES of 640 by one
// 640-thread CTA (quadmp_schedule.hpp):
//   phase 0      positions x + (xl + d) of ALL vertices -> shared memory (coloured slots), accumulators zeroed
//   sweep        unit normals of ALL triangles -> shared memory, 6V by fixed-point REDUX + shared atomics
//   pass 0 .. 3  the pass's 29 per-quad words come from L2 into registers (the next pass's loads are in flight while
//                the vertices gather); membrane, five hinges, four corner-force stores into the pass's slots; then the
//                vertices the pass touches (its list) gather their slots and add them to per-vertex accumulators
//   phase C      r = coef d - b + accumulator -> global
// Replaces local_big.cu's 1024-thread kernel (tables streamed per triangle, corner forces in chunks, 42 % bank-conflict
// wavefronts): here every gather is coloured conflict-free or nearly so, exactly as in the one-pass kernel.
// Shared memory for RBC-2562: positions 41 KB + normals 82 KB + corner forces of one pass 41 KB + accumulators 31 KB.
#include "internal.h"

namespace npfem {
namespace {

constexpr int QW = 7, QK = 22, TH = 640;
constexpr int NP = 4;    // passes at most (QMP_MAX_PASSES)
constexpr int NV = 5;    // vertices per thread at most: n <= NP * TH + 2

struct QuadMpParams {
  int n, n_pad, nq, passes, lstride;
  int list_len[4];
  int sx_bytes, sN_bytes, sC_bytes;
  const uint32_t *quad_words;   // [passes][QW][TH] slot INDICES, 16 bit each
  const float *quad_consts;     // [passes][QK][TH]
  const uint32_t *list_words;   // [passes][1 + MAXV/2][lstride]
  const uint32_t *vtx_slot;     // [n]
  const float *vtx_coef;        // [n]
  float fx_scale;
  long long fx_rest;
  float vc_scale;
  const float *x, *xl, *d, *b;  // [cells][3][n_pad]
  float *g;
  int g_tf32;
  int64_t cells;
};

__device__ __forceinline__ float rsqrt_fast(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ uint32_t lo16(uint32_t w) {
  uint32_t r;
  asm volatile("and.b32 %0, %1, 0xffff;" : "=r"(r) : "r"(w));
  return r;
}
__device__ __forceinline__ uint32_t hi16(uint32_t w) {
  uint32_t r;
  asm volatile("shr.u32 %0, %1, 16;" : "=r"(r) : "r"(w));
  return r;
}
__device__ __forceinline__ float4 lds4(const unsigned char *base, uint32_t off) {
  return *reinterpret_cast<const float4 *>(base + off);
}
__device__ __forceinline__ void sts4(unsigned char *base, uint32_t off, float x, float y, float z, float w) {
  *reinterpret_cast<float4 *>(base + off) = make_float4(x, y, z, w);
}

// NPAD: compile-time row pitch of the state fields (0 = run-time p.n_pad): loads of a thread's vertices then share one
// base register per field
template <int MAXV, int NPAD>
__global__ void __launch_bounds__(TH, 1) local_quadmp_kernel(const QuadMpParams p) {
  extern __shared__ __align__(16) unsigned char smem[];
  constexpr int VWORDS = 1 + MAXV / 2;
  const int n = p.n, n_pad = NPAD ? NPAD : p.n_pad;
  unsigned char *sx = smem;
  unsigned char *sN = sx + p.sx_bytes;
  unsigned char *sC = sN + p.sN_bytes;
  float *acc = reinterpret_cast<float *>(sC + p.sC_bytes);     // [3][n_pad] corner-force sums per vertex
  int *vacc = reinterpret_cast<int *>(acc + 3 * n_pad);        // [hi, lo] base-2^12 digits of 6V (fixed point)
  uint64_t *bar_acc = reinterpret_cast<uint64_t *>(vacc + 2);  // split barrier "accumulators of the pass updated"
  const int tid = threadIdx.x, lane = tid & 31;

  if (tid < 8) sts4(sC, uint32_t(p.sC_bytes) - 128u + 16u * tid, 0.f, 0.f, 0.f, 0.f);   // the zero slots
  if (tid == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(uint32_t(__cvta_generic_to_shared(bar_acc))), "r"(TH / 32));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  // arrive early (after the pass's accumulation), wait late (before the next corner-force stores / before phase C):
  // the threads with two list entries no longer hold up the others at a second block barrier per pass
  auto acc_arrive = [&]() {
    __syncwarp();
    if (lane == 0)
      asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(uint32_t(__cvta_generic_to_shared(bar_acc))) : "memory");
  };
  auto acc_wait = [&](uint32_t parity) {
    uint32_t done;
    do {
      asm volatile(
          "{\n.reg .pred q;\nmbarrier.try_wait.parity.shared::cta.b64 q, [%1], %2, %3;\nselp.u32 %0, 1, 0, q;\n}\n"
          : "=r"(done) : "r"(uint32_t(__cvta_generic_to_shared(bar_acc))), "r"(parity), "r"(20000u) : "memory");
    } while (!done);
  };
  uint32_t acc_phase = 0;      // completed phases of bar_acc (one per pass)
  uint32_t qw[QW];
  float qk[QK];
  auto load_pass = [&](int ps) {   // this thread's quad of pass ps (zeros beyond the last quad: nothing is stored then)
    const bool a = ps * TH + tid < p.nq;
#pragma unroll
    for (int q = 0; q < QW; ++q) qw[q] = a ? __ldg(p.quad_words + (ps * QW + q) * TH + tid) : 0u;
#pragma unroll
    for (int q = 0; q < QK; ++q) qk[q] = a ? __ldg(p.quad_consts + (ps * QK + q) * TH + tid) : 0.f;
  };

  for (int64_t cell = blockIdx.x; cell < p.cells; cell += gridDim.x) {
    const size_t base = size_t(cell) * 3 * n_pad;
    // the sweep's table words first: their L2 latency runs under phase 0
    uint32_t w0[NP], w1[NP], w4[NP];
#pragma unroll
    for (int ps = 0; ps < NP; ++ps) {
      const bool a = ps < p.passes && ps * TH + tid < p.nq;
      w0[ps] = a ? __ldg(p.quad_words + (ps * QW + 0) * TH + tid) : 0u;
      w1[ps] = a ? __ldg(p.quad_words + (ps * QW + 1) * TH + tid) : 0u;
      w4[ps] = a ? __ldg(p.quad_words + (ps * QW + 4) * TH + tid) : 0u;
    }
    // ---- phase 0: current positions from the two-float x_n = x + xl, accumulators ------------------------------
    if (tid == 0) vacc[0] = vacc[1] = 0;
    // (in batches of three vertices per thread: all loads of a batch in flight together)
#pragma unroll
    for (int j0 = 0; j0 < NV; j0 += 3) {
      float px[3][3];
      uint32_t sl[3];
#pragma unroll
      for (int jj = 0; jj < 3; ++jj) {
        const int v = tid + (j0 + jj) * TH;
        const bool a = j0 + jj < NV && v < n;
        const float *x = p.x + base + v, *xl = p.xl + base + v, *d = p.d + base + v;
        sl[jj] = a ? __ldg(p.vtx_slot + v) : 0u;
#pragma unroll
        for (int c = 0; c < 3; ++c)
          px[jj][c] = a ? __ldcs(x + c * n_pad) + (__ldcs(xl + c * n_pad) + __ldcs(d + c * n_pad)) : 0.f;
      }
#pragma unroll
      for (int jj = 0; jj < 3; ++jj) {
        const int v = tid + (j0 + jj) * TH;
        if (j0 + jj < NV && v < n) {
          sts4(sx, sl[jj] << 4, px[jj][0], px[jj][1], px[jj][2], 0.f);
          acc[v] = 0.f;
          acc[n_pad + v] = 0.f;
          acc[2 * n_pad + v] = 0.f;
        }
      }
    }
    // the next cell's x, xl, d, b on their way into L2 while this one is computed (phase 0 / phase C then see L2
    // latency instead of DRAM latency: one 640-thread CTA has too few loads in flight to hide the latter)
    if (cell + gridDim.x < p.cells) {
      const size_t nb = size_t(cell + gridDim.x) * 3 * n_pad;
      const int lines = (3 * n_pad * 4 + 127) / 128;
      for (int l = tid; l < 4 * lines; l += TH) {
        const float *f = l < lines ? p.x : (l < 2 * lines ? p.xl : (l < 3 * lines ? p.d : p.b));
        const char *ptr = reinterpret_cast<const char *>(f + nb) + size_t(l % lines) * 128;
        asm volatile("prefetch.global.L2 [%0];" ::"l"(ptr));
      }
    }
    __syncthreads();
    // ---- sweep: unit normals of all triangles, 6V ---------------------------------------------------------------
    {
      float vol = 0.f;
#pragma unroll
      for (int ps = 0; ps < NP; ++ps) {
        if (ps < p.passes && ps * TH + tid < p.nq) {
          const float4 Xp = lds4(sx, (w0[ps] & 0xffffu) << 4), Xq = lds4(sx, (w0[ps] >> 16) << 4),
                       Xr = lds4(sx, (w1[ps] & 0xffffu) << 4), Xs = lds4(sx, (w1[ps] >> 16) << 4);
          const float a0 = Xq.x - Xp.x, a1 = Xq.y - Xp.y, a2 = Xq.z - Xp.z;       // e1
          const float b0 = Xr.x - Xp.x, b1 = Xr.y - Xp.y, b2 = Xr.z - Xp.z;       // e2
          const float c0 = Xs.x - Xp.x, c1 = Xs.y - Xp.y, c2 = Xs.z - Xp.z;       // f
          const float N0x = a1 * b2 - a2 * b1, N0y = a2 * b0 - a0 * b2, N0z = a0 * b1 - a1 * b0;   // T0: e1 x e2
          const float N1x = c1 * a2 - c2 * a1, N1y = c2 * a0 - c0 * a2, N1z = c0 * a1 - c1 * a0;   // T1: f x e1
          const float i0 = rsqrt_fast(N0x * N0x + N0y * N0y + N0z * N0z), i1 = rsqrt_fast(N1x * N1x + N1y * N1y + N1z * N1z);
          // 6 x signed tetrahedron volumes of both triangles (both have p as their first corner)
          vol += Xp.x * (N0x + N1x) + Xp.y * (N0y + N1y) + Xp.z * (N0z + N1z);
          sts4(sN, (w4[ps] & 0xffffu) << 4, N0x * i0, N0y * i0, N0z * i0, i0);
          sts4(sN, (w4[ps] >> 16) << 4, N1x * i1, N1y * i1, N1z * i1, i1);
        }
        if (ps == 1) load_pass(0);     // the first pass's 29 words: requested half way through the sweep
      }
      // fixed point as in local_quad.cu: one REDUX, integer shared atomics, exact and order independent
      const int wsum = __reduce_add_sync(0xffffffffu, __float2int_rn(vol * p.fx_scale));
      if (lane == 0) {
        atomicAdd(vacc, wsum >> 12);          // signed high digit
        atomicAdd(vacc + 1, wsum & 0xfff);    // 12-bit low digit
      }
    }
    __syncthreads();
    // (the cast to int is the modular reduction that makes the fixed-point difference exact: local_quad.cu)
    const float vc = p.vc_scale * float(int((static_cast<long long>(vacc[0]) << 12) + vacc[1] - p.fx_rest));
    // ---- the passes ---------------------------------------------------------------------------------------------
    for (int ps = 0; ps < p.passes; ++ps) {
      const bool act = ps * TH + tid < p.nq;
      {
        // ---- the four vertices and both normals again (registers only; cheaper than keeping them across the sweep) ----
      float e1[3], e2[3], f[3], n0[3], n1[3], inv0, inv1, nn0, nn1;
      {
        const float4 Xp = lds4(sx, (lo16(qw[0]) << 4)), Xq = lds4(sx, (hi16(qw[0]) << 4)), Xr = lds4(sx, (lo16(qw[1]) << 4)), Xs = lds4(sx, (hi16(qw[1]) << 4));
        e1[0] = Xq.x - Xp.x; e1[1] = Xq.y - Xp.y; e1[2] = Xq.z - Xp.z;
        e2[0] = Xr.x - Xp.x; e2[1] = Xr.y - Xp.y; e2[2] = Xr.z - Xp.z;
        f[0] = Xs.x - Xp.x; f[1] = Xs.y - Xp.y; f[2] = Xs.z - Xp.z;
        // T0 = (p, q, r): N0 = e1 x e2;  T1 = (p, s, q): N1 = f x e1
        const float N0x = e1[1] * e2[2] - e1[2] * e2[1], N0y = e1[2] * e2[0] - e1[0] * e2[2], N0z = e1[0] * e2[1] - e1[1] * e2[0];
        const float N1x = f[1] * e1[2] - f[2] * e1[1], N1y = f[2] * e1[0] - f[0] * e1[2], N1z = f[0] * e1[1] - f[1] * e1[0];
        nn0 = N0x * N0x + N0y * N0y + N0z * N0z;
        nn1 = N1x * N1x + N1y * N1y + N1z * N1z;
        inv0 = rsqrt_fast(nn0);
        inv1 = rsqrt_fast(nn1);
        n0[0] = N0x * inv0; n0[1] = N0y * inv0; n0[2] = N0z * inv0;
        n1[0] = N1x * inv1; n1[1] = N1y * inv1; n1[2] = N1z * inv1;
      }
      // (Skalak, readings R5/R7): Q = 2 A0 (W1 R + W2 det^2 adj G)
      // T0 with edges (e1, e2), T1 with edges (f, e1): |e1|^2 is shared
      const float e11 = e1[0] * e1[0] + e1[1] * e1[1] + e1[2] * e1[2];
      const float e12 = e1[0] * e2[0] + e1[1] * e2[1] + e1[2] * e2[2];
      const float e22 = e2[0] * e2[0] + e2[1] * e2[1] + e2[2] * e2[2];
      const float ff = f[0] * f[0] + f[1] * f[1] + f[2] * f[2];
      const float fe = f[0] * e1[0] + f[1] * e1[1] + f[2] * e1[2];
      float q11, q12, q22, r11, r12, r22;               // Q of T0 and of T1
      {
        const float R11 = qk[0], R12 = qk[1], R22 = qk[2], J = qk[3], tA = qk[4], tC = qk[5];
        const float th = fmaf(R12, e12, -0.5f);
        const float I1p1 = fmaf(R11, e11, fmaf(R22, e22, th + th));            // I1 + 1
        const float I2 = fmaf(J, nn0, -1.f);
        const float W1 = tA * I1p1, W2 = fmaf(tC, I2, -tA * J);
        q11 = fmaf(W2, e22, W1 * R11);
        q22 = fmaf(W2, e11, W1 * R22);
        q12 = fmaf(-W2, e12, W1 * R12);
      }
      {
        const float R11 = qk[6], R12 = qk[7], R22 = qk[8], J = qk[9], tA = qk[10], tC = qk[11];
        const float th = fmaf(R12, fe, -0.5f);
        const float I1p1 = fmaf(R11, ff, fmaf(R22, e11, th + th));
        const float I2 = fmaf(J, nn1, -1.f);
        const float W1 = tA * I1p1, W2 = fmaf(tC, I2, -tA * J);
        r11 = fmaf(W2, e11, W1 * R11);
        r22 = fmaf(W2, ff, W1 * R22);
        r12 = fmaf(-W2, fe, W1 * R12);
      }
      // hinge weights on the corners of T0 = (p, q, r): w0..w2, and of T1 = (p, s, q): z0..z2 (reading R8; side k of a
      // triangle with edges (a1, a2) runs from corner k to k+1: a1, a2 - a1, -a2)
      float w0, w1, w2, z0, z1, z2;
      {   // shared hinge p-q: side 0 of T0 (neighbour normal n1), side 2 of T1 (neighbour normal n0): ONE scalar
        const float crx = n0[1] * n1[2] - n0[2] * n1[1], cry = n0[2] * n1[0] - n0[0] * n1[2], crz = n0[0] * n1[1] - n0[1] * n1[0];
        const float S = crx * e1[0] + cry * e1[1] + crz * e1[2];
        const float cs = n0[0] * n1[0] + n0[1] * n1[1] + n0[2] * n1[2];
        const float L = e11, ie = rsqrt_fast(L);
        const float q = ie * fmaf(S * ie, qk[12], -cs * qk[17]);   // dE/dtheta / |e|
        const float D = e11 - e12;                                 // T0, side 0
        w0 = D * q; w1 = (L - D) * q; w2 = -L * q;
        z2 = fe * q; z0 = (L - fe) * q; z1 = -L * q;               // T1, side 2: L = |a2|^2 = e11, D = a1 . a2 = fe
      }
      // ---- phase B ----------------------------------------------------------------------------
      // the four neighbour normals first (independent loads in flight together), then the five hinges
      const float4 NB0 = lds4(sN, (lo16(qw[2]) << 4)), NB1 = lds4(sN, (hi16(qw[2]) << 4)), NB2 = lds4(sN, (lo16(qw[3]) << 4)), NB3 = lds4(sN, (hi16(qw[3]) << 4));
      {   // T0 side 1: q -> r, neighbour NB0
        const float4 B = NB0;
        const float crx = n0[1] * B.z - n0[2] * B.y, cry = n0[2] * B.x - n0[0] * B.z, crz = n0[0] * B.y - n0[1] * B.x;
        const float S = crx * (e2[0] - e1[0]) + cry * (e2[1] - e1[1]) + crz * (e2[2] - e1[2]);
        const float cs = n0[0] * B.x + n0[1] * B.y + n0[2] * B.z;
        const float L = e11 - 2.f * e12 + e22, D = e22 - e12, ie = rsqrt_fast(L);
        const float q = ie * fmaf(S * ie, qk[13], -cs * qk[18]);
        w1 = fmaf(D, q, w1); w2 = fmaf(L - D, q, w2); w0 = fmaf(-L, q, w0);
      }
      {   // T0 side 2: r -> p, neighbour NB1
        const float4 B = NB1;
        const float crx = n0[1] * B.z - n0[2] * B.y, cry = n0[2] * B.x - n0[0] * B.z, crz = n0[0] * B.y - n0[1] * B.x;
        const float S = -(crx * e2[0] + cry * e2[1] + crz * e2[2]);
        const float cs = n0[0] * B.x + n0[1] * B.y + n0[2] * B.z;
        const float L = e22, D = e12, ie = rsqrt_fast(L);
        const float q = ie * fmaf(S * ie, qk[14], -cs * qk[19]);
        w2 = fmaf(D, q, w2); w0 = fmaf(L - D, q, w0); w1 = fmaf(-L, q, w1);
      }
      {   // T1 side 0: p -> s (edge a1 = f), neighbour NB2
        const float4 B = NB2;
        const float crx = n1[1] * B.z - n1[2] * B.y, cry = n1[2] * B.x - n1[0] * B.z, crz = n1[0] * B.y - n1[1] * B.x;
        const float S = crx * f[0] + cry * f[1] + crz * f[2];
        const float cs = n1[0] * B.x + n1[1] * B.y + n1[2] * B.z;
        const float L = ff, D = ff - fe, ie = rsqrt_fast(L);
        const float q = ie * fmaf(S * ie, qk[15], -cs * qk[20]);
        z0 = fmaf(D, q, z0); z1 = fmaf(L - D, q, z1); z2 = fmaf(-L, q, z2);
      }
      {   // T1 side 1: s -> q (edge a2 - a1 = e1 - f), neighbour NB3
        const float4 B = NB3;
        const float crx = n1[1] * B.z - n1[2] * B.y, cry = n1[2] * B.x - n1[0] * B.z, crz = n1[0] * B.y - n1[1] * B.x;
        const float S = crx * (e1[0] - f[0]) + cry * (e1[1] - f[1]) + crz * (e1[2] - f[2]);
        const float cs = n1[0] * B.x + n1[1] * B.y + n1[2] * B.z;
        const float L = ff - 2.f * fe + e11, D = e11 - fe, ie = rsqrt_fast(L);
        const float q = ie * fmaf(S * ie, qk[16], -cs * qk[21]);
        z1 = fmaf(D, q, z1); z2 = fmaf(L - D, q, z2); z0 = fmaf(-L, q, z0);
      }
      // corner forces: volume term (reading R9) + hinge terms along the unit normals + membrane; the two triangles'
      // forces on p and on q are summed here, so the quad stores FOUR vectors
      float cp[3], cq[3], cr[3], cs4[3];
      {
        const float vn0 = vc * (nn0 * inv0), vn1 = vc * (nn1 * inv1);
        const float u0 = fmaf(inv0, w0, vn0), u1 = fmaf(inv0, w1, vn0), u2 = fmaf(inv0, w2, vn0), us = u0 + u1 + u2;
        const float y0 = fmaf(inv1, z0, vn1), y1 = fmaf(inv1, z1, vn1), y2 = fmaf(inv1, z2, vn1), ys = y0 + y1 + y2;
  #pragma unroll
        for (int k = 0; k < 3; ++k) {
          const float c1 = fmaf(u1, n0[k], fmaf(q11, e1[k], q12 * e2[k]));      // T0 corner q
          const float c2 = fmaf(u2, n0[k], fmaf(q12, e1[k], q22 * e2[k]));      // T0 corner r
          const float c0 = fmaf(us, n0[k], -c1) - c2;                            // T0 corner p
          const float t1 = fmaf(y1, n1[k], fmaf(r11, f[k], r12 * e1[k]));       // T1 corner s
          const float t2 = fmaf(y2, n1[k], fmaf(r12, f[k], r22 * e1[k]));       // T1 corner q
          const float t0 = fmaf(ys, n1[k], -t1) - t2;                            // T1 corner p
          cp[k] = c0 + t0;
          cq[k] = c1 + t2;
          cr[k] = c2;
          cs4[k] = t1;
        }
      }
      if (ps > 0) acc_wait((acc_phase - 1) & 1u);     // the previous pass's gathers from sC are done
      if (act) {
        sts4(sC, (lo16(qw[5]) << 4), cp[0], cp[1], cp[2], 0.f);
        sts4(sC, (hi16(qw[5]) << 4), cq[0], cq[1], cq[2], 0.f);
        sts4(sC, (lo16(qw[6]) << 4), cr[0], cr[1], cr[2], 0.f);
        sts4(sC, (hi16(qw[6]) << 4), cs4[0], cs4[1], cs4[2], 0.f);
      }
      }
      if (ps + 1 < p.passes) load_pass(ps + 1);       // in flight during the barrier and the gathers below
      // this thread's (at most two) entries of the pass's vertex list: loaded in front of the barrier as well
      uint32_t lw[2][VWORDS];
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        const int e = tid + j * TH;
        const uint32_t *src = p.list_words + size_t(ps * VWORDS) * p.lstride + e;
#pragma unroll
        for (int q = 0; q < VWORDS; ++q) lw[j][q] = e < p.list_len[ps] ? __ldg(src + q * p.lstride) : 0u;
      }
      __syncthreads();
      // the vertices this pass touches add their corner forces to their accumulators (one thread per vertex and pass)
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        if (tid + j * TH < p.list_len[ps]) {
          const uint32_t vid = lw[j][0];
          float4 f[MAXV];
#pragma unroll
          for (int q = 0; q < MAXV; q += 2) {
            const uint32_t w = lw[j][1 + (q >> 1)];
            f[q] = lds4(sC, (w & 0xffffu) << 4);
            f[q + 1] = lds4(sC, (w >> 16) << 4);
          }
          float ax = 0.f, ay = 0.f, az = 0.f;
#pragma unroll
          for (int q = 0; q < MAXV; ++q) { ax += f[q].x; ay += f[q].y; az += f[q].z; }
          acc[vid] += ax;
          acc[n_pad + vid] += ay;
          acc[2 * n_pad + vid] += az;
        }
      }
      acc_arrive();
      ++acc_phase;
    }
    // ---- phase C: r = coef d - b + the vertex's corner forces -> global -----------------------------------------
    // (merging it with phase 0 of the CTA's next cell, loads of both issued together, was tried: 0.99 vs 0.94 ms)
#pragma unroll
    for (int j0 = 0; j0 < NV; j0 += 3) {
      float dd[3][3], bb[3][3], coef[3];
#pragma unroll
      for (int jj = 0; jj < 3; ++jj) {
        const int v = tid + (j0 + jj) * TH;
        const bool a = j0 + jj < NV && v < n;
        coef[jj] = a ? __ldg(p.vtx_coef + v) : 0.f;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          dd[jj][c] = a ? __ldcs(p.d + base + c * n_pad + v) : 0.f;
          bb[jj][c] = a ? __ldcs(p.b + base + c * n_pad + v) : 0.f;
        }
      }
      if (j0 == 0) acc_wait((acc_phase - 1) & 1u);    // every accumulator is final (the loads above are in flight)
#pragma unroll
      for (int jj = 0; jj < 3; ++jj) {
        const int v = tid + (j0 + jj) * TH;
        if (j0 + jj < NV && v < n) {
          float g0 = fmaf(coef[jj], dd[jj][0], acc[v] - bb[jj][0]);
          float g1 = fmaf(coef[jj], dd[jj][1], acc[n_pad + v] - bb[jj][1]);
          float g2 = fmaf(coef[jj], dd[jj][2], acc[2 * n_pad + v] - bb[jj][2]);
          if (p.g_tf32) { g0 = tf32_rn(g0); g1 = tf32_rn(g1); g2 = tf32_rn(g2); }
          float *gout = p.g + base + v;
          gout[0] = g0;
          gout[n_pad] = g1;
          gout[2 * n_pad] = g2;
        }
      }
    }
    // the next cell's phase 0 rewrites sx (last read in the last pass's arithmetic, which every warp has left: the wait
    // above) and zeroes acc[v] in the thread that has just read it
  }
}

size_t quadmp_smem_bytes(const QuadMpDev &s, int n_pad) {
  return size_t(s.n_vslots + s.n_tslots + s.n_cslots) * 16 + size_t(3) * n_pad * 4 + 8 + 8;
}

}  // namespace

bool local_quadmp_supported(const TypeDev &td) {
  const QuadMpDev &s = td.quadmp;
  return s.valid && s.passes >= 1 && s.passes <= 4 && (s.maxv == 6 || s.maxv == 8) && quadmp_smem_bytes(s, td.n_pad) <= 227 * 1024;
}

int launch_local_quadmp(const TypeDev &td, const BucketView &bv, int n_sm, cudaStream_t stream) {
  if (bv.cells == 0) return 0;
  if (!local_quadmp_supported(td)) return -1;
  const QuadMpDev &s = td.quadmp;
  QuadMpParams p;
  p.n = td.n; p.n_pad = td.n_pad; p.nq = s.nq; p.passes = s.passes; p.lstride = s.lstride;
  for (int i = 0; i < 4; ++i) p.list_len[i] = s.list_len[i];
  p.sx_bytes = s.n_vslots * 16; p.sN_bytes = s.n_tslots * 16; p.sC_bytes = s.n_cslots * 16;
  p.quad_words = s.quad_words; p.quad_consts = s.quad_consts; p.list_words = s.list_words;
  p.vtx_slot = s.vtx_slot; p.vtx_coef = s.vtx_coef;
  // fixed-point 6V: 32 lane partials (one quad per pass each) with 16 x headroom over the rest shape
  int k = 0;
  std::frexp(16.0 * 32.0 * s.vol_lane_bound, &k);
  const double scale = std::ldexp(1.0, 31 - k);
  p.fx_scale = float(scale);
  p.fx_rest = std::llrint(6.0 * td.V0 * scale);
  p.vc_scale = float(td.kv_over_V0 / 36.0 / scale);
  p.x = static_cast<const float *>(bv.field[F_X]);
  p.xl = static_cast<const float *>(bv.field[F_XL]);
  p.d = static_cast<const float *>(bv.field[F_D]);
  p.b = static_cast<const float *>(bv.field[F_B]);
  p.g = static_cast<float *>(bv.field[F_G]);
  p.g_tf32 = bv.g_tf32;
  p.cells = bv.cells;
  const size_t smem = quadmp_smem_bytes(s, td.n_pad);
  const int64_t grid = bv.cells < n_sm ? bv.cells : n_sm;       // one CTA per SM (shared memory and registers)
  auto go = [&](auto kernel) {
    if (!td.cache.quadmp_attr && opt_in_max_dynamic_smem(kernel) != cudaSuccess) return -1;
    td.cache.quadmp_attr = true;
    kernel<<<unsigned(grid), TH, smem, stream>>>(p);
    return 1;
  };
  if (s.maxv == 6) return td.n_pad == 2576 ? go(local_quadmp_kernel<6, 2576>) : go(local_quadmp_kernel<6, 0>);
  return go(local_quadmp_kernel<8, 0>);
}

}  // namespace npfem
