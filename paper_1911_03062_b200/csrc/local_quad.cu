// Local step (row a2), fp32 "quad" path: the scheduled kernel of local_sched.cu with ONE THREAD PER PAIR OF ADJACENT
// TRIANGLES  T0 = (p, q, r), T1 = (p, s, q)  (shared edge p-q; quad_schedule.hpp finds the pairing, a perfect matching
// of the dual graph, and the conflict-free shared-memory slots).  Same reduced gradient
//   r = (1 - gamma) m^ d - b + grad E(x_n + d)     (Eqs. (3)-(4), energies = readings R5-R9)
// same staging ring, split barriers and fixed-point volume; what changes is the work per cell:
//   * 4 vertex gathers and 4 neighbour-normal gathers per thread instead of 6 + 6 (p, q and the normals of T0 / T1
//     are shared inside the thread);
//   * the shared hinge p-q is evaluated once (its scalar dE/dtheta / |e| serves both triangles);
//   * the two triangles' forces on p and on q are summed in registers: 4 corner-force stores instead of 6, and a
//     vertex gathers one slot per incident quad (4 on average, at most 6) instead of one per incident triangle;
//   * 29 instead of 34 constant registers per thread.
#include "internal.h"

namespace npfem {
namespace {

constexpr int NSTAGE = 3;
constexpr int QW = 7, QK = 22;   // packed offset words / float constants per quad (quad_schedule.hpp)

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return uint32_t(__cvta_generic_to_shared(p)); }

struct QuadParams {
  int n, T, n_pad, ttri, threads, vstride;   // T = quads, ttri = threads that own a quad slot
  int sx_bytes, sN_bytes, sC_bytes;
  const uint32_t *tri_words;   // [QW][threads]
  const float *tri_consts;     // [QK][threads]
  const uint32_t *vtx_words;   // [1 + MAXV/2][vstride]
  const float *vtx_coef;       // [vstride]
  float fx_scale;              // per-lane 6V partials are reduced as integers in units of 1 / fx_scale
  long long fx_rest;           // round(6 V0 fx_scale)
  float vc_scale;              // k_v / (36 V0) / fx_scale:  vc = vc_scale (6V - 6V0)_fixed = k_v (V - V0)/V0 / 6
  const float *x, *xl, *d, *b; // [cells][3][n_pad]; the position of a vertex is x + xl (two-float, internal.h F_XL)
  float *g;
  int g_tf32;                  // round g to TF32 (its consumer is the tensor-core GEMM)
  int64_t cells;
};

// plain MUFU.RSQ: no denormal rescue (squared edge lengths / areas of a live mesh are normal numbers)
__device__ __forceinline__ float rsqrt_fast(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// 16-bit halves of a packed offset word.  volatile: re-extracted at every use instead of being kept
// unpacked in registers for the whole launch (the register budget is what limits this kernel)
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

// NPAD: compile-time row pitch of the state fields (0 = run-time p.n_pad): with it every access to the
// staging ring is base register + immediate instead of a per-access address computation
template <int MAXV, int MAXT, int MINB, int NPAD>
__global__ void __launch_bounds__(MAXT, MINB) local_quad_kernel(const QuadParams p) {
  extern __shared__ __align__(16) unsigned char smem[];
  const int n = p.n, n_pad = NPAD ? NPAD : p.n_pad, nthreads = p.threads;
  unsigned char *sx = smem;
  unsigned char *sN = sx + p.sx_bytes;
  unsigned char *sC = sN + p.sN_bytes;
  float *stage = reinterpret_cast<float *>(sC + p.sC_bytes);            // [NSTAGE][4 fields x, d, b, xl][3][n_pad]
  int *vacc = reinterpret_cast<int *>(stage + NSTAGE * 12 * n_pad);   // [2 cells][hi, lo] base-2^12 digits of 6V (fixed point)
  uint64_t *mbar = reinterpret_cast<uint64_t *>(vacc + 4);   // [NSTAGE] TMA ring
  uint64_t *bars = mbar + NSTAGE;                              // [4] split block barriers B1, B2, B3, BV

  const int tid = threadIdx.x, lane = tid & 31;
  const uint32_t field_bytes = uint32_t(3 * n_pad) * 4u;

  // ---- per-thread constants: registers for the whole launch ---------------------------------
  // qw: 0 = p | q, 1 = r | s (vertex slots), 2 = n0 | n1 (normals across q-r, r-p), 3 = n2 | n3 (across p-s, s-q),
  //     4 = own normal slots T0 | T1, 5 = corner slots p | q, 6 = r | s          (16-bit byte offsets)
  // qk: 0..5 = R11 R12 R22 J tA tC of T0 = (p, q, r), 6..11 = of T1 = (p, s, q), 12..16 = k_b cos theta0 and
  //     17..21 = k_b sin theta0 of the hinges  shared p-q, q-r, r-p, p-s, s-q
  uint32_t qw[QW];
  float qk[QK];
  const bool act = tid < p.T;
#pragma unroll
  for (int q = 0; q < QW; ++q) qw[q] = p.tri_words[q * nthreads + tid];
#pragma unroll
  for (int q = 0; q < QK; ++q) qk[q] = p.tri_consts[q * nthreads + tid];
  uint32_t vw[1 + MAXV / 2];
#pragma unroll
  for (int q = 0; q < 1 + MAXV / 2; ++q) vw[q] = p.vtx_words[q * p.vstride + tid];
  const float coef = p.vtx_coef[tid];
  const bool vact = tid < n;
  // a few vertices may need a second pass (n slightly above the CTA size): the LAST warp takes them
  // (warp 0 already issues the TMA prefetches: any extra work of ONE warp delays the whole block at
  // the next barrier), their constants stay in global memory (L1 hits)
  // phase 0 of the overflow vertices runs in the last warp, their phase C in the one before it, so
  // no warp carries both extras
  const int v2 = tid + 32;
  const bool vact2 = tid >= nthreads - 32 && v2 < n;
  const int v2c = tid + 64;
  const bool vact2c = tid >= nthreads - 64 && tid < nthreads - 32 && v2c < n;

  auto prefetch = [&](int64_t cell, int st) {   // one thread: arm the barrier, start 4 bulk copies
    const size_t base = size_t(cell) * 3 * n_pad;
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(mbar + st)),
                 "r"(4u * field_bytes) : "memory");
    const float *src[4] = {p.x + base, p.d + base, p.b + base, p.xl + base};
#pragma unroll
    for (int f = 0; f < 4; ++f)
      asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                   ::"r"(smem_u32(stage + (st * 12 + f * 3) * n_pad)), "l"(src[f]), "r"(field_bytes),
                     "r"(smem_u32(mbar + st)) : "memory");
  };

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NSTAGE; ++s) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(mbar + s)));
#pragma unroll
    for (int s = 0; s < 4; ++s)
      asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bars + s)), "r"(nthreads >> 5));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    vacc[0] = vacc[1] = vacc[2] = vacc[3] = 0;
  }
  if (tid < 8) sts4(sC, uint32_t(p.sC_bytes) - 128u + 16u * tid, 0.f, 0.f, 0.f, 0.f);   // the zero slots
  __syncthreads();
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NSTAGE - 1; ++s) {
      const int64_t c = int64_t(blockIdx.x) + int64_t(s) * gridDim.x;
      if (c < p.cells) prefetch(c, s);
    }
  }

  // block-wide split barriers (arrive early, wait late) on mbarriers, one arrival per warp
  auto bar_arrive = [&](int which) {
    __syncwarp();
    if (lane == 0)
      asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bars + which)) : "memory");
  };
  auto bar_wait = [&](int which, uint32_t parity) {
    uint32_t done;
    do {
      asm volatile(
          "{\n.reg .pred q;\nmbarrier.try_wait.parity.shared::cta.b64 q, [%1], %2, %3;\nselp.u32 %0, 1, 0, q;\n}\n"
          : "=r"(done) : "r"(smem_u32(bars + which)), "r"(parity), "r"(20000u) : "memory");   // suspend-time hint, ns
    } while (!done);
  };
  // phase 0 of this CTA's it0-th cell (ring slot it0 % NSTAGE): sx[slot(v)] = (x + (xl + d), 0), the current
  // position from the two-float x_n = x + xl
  auto phase0_vertex = [&](const float *sg, int v, uint32_t slot_off) {
    sts4(sx, slot_off, sg[v] + (sg[9 * n_pad + v] + sg[3 * n_pad + v]),
         sg[n_pad + v] + (sg[10 * n_pad + v] + sg[4 * n_pad + v]),
         sg[2 * n_pad + v] + (sg[11 * n_pad + v] + sg[5 * n_pad + v]), 0.f);
  };
  auto phase0 = [&](int it0) {
    const int st = it0 % NSTAGE;
    const float *sg = stage + st * 12 * n_pad;
    const uint32_t parity = uint32_t(it0 / NSTAGE) & 1u;
    uint32_t done;
    do {
      asm volatile(
          "{\n.reg .pred q;\nmbarrier.try_wait.parity.shared::cta.b64 q, [%1], %2;\nselp.u32 %0, 1, 0, q;\n}\n"
          : "=r"(done) : "r"(smem_u32(mbar + st)), "r"(parity) : "memory");
    } while (!done);
    if (vact) phase0_vertex(sg, tid, lo16(vw[0]));
    if (vact2) phase0_vertex(sg, v2, p.vtx_words[v2] & 0xffffu);
  };

  // ---- phase C of one cell: r = coef d - b + sum of the vertex's corner forces -> global ---------------
  auto phaseC = [&](int64_t cell, const float *sg) {
    if (vact) {
      float4 f[MAXV];
#pragma unroll
      for (int q = 0; q < MAXV; ++q)
        f[q] = lds4(sC, (q & 1) ? hi16(vw[1 + (q >> 1)]) : lo16(vw[1 + (q >> 1)]));
      float ax = 0.f, ay = 0.f, az = 0.f;
#pragma unroll
      for (int q = 0; q < MAXV; ++q) { ax += f[q].x; ay += f[q].y; az += f[q].z; }
      float *gout = p.g + size_t(cell) * 3 * n_pad + tid;
      float g0 = fmaf(coef, sg[3 * n_pad + tid], ax - sg[6 * n_pad + tid]);
      float g1 = fmaf(coef, sg[4 * n_pad + tid], ay - sg[7 * n_pad + tid]);
      float g2 = fmaf(coef, sg[5 * n_pad + tid], az - sg[8 * n_pad + tid]);
      if (p.g_tf32) { g0 = tf32_rn(g0); g1 = tf32_rn(g1); g2 = tf32_rn(g2); }
      gout[0] = g0;
      gout[n_pad] = g1;
      gout[2 * n_pad] = g2;
    }
    if (vact2c) {
      float ax = 0.f, ay = 0.f, az = 0.f;
      for (int q = 0; q < MAXV; ++q) {
        const uint32_t w = p.vtx_words[(1 + (q >> 1)) * p.vstride + v2c];
        const float4 f = lds4(sC, (q & 1) ? (w >> 16) : (w & 0xffffu));
        ax += f.x; ay += f.y; az += f.z;
      }
      const float coef2 = p.vtx_coef[v2c];
      float *gout = p.g + size_t(cell) * 3 * n_pad + v2c;
      const float g0 = fmaf(coef2, sg[3 * n_pad + v2c], ax - sg[6 * n_pad + v2c]);
      const float g1 = fmaf(coef2, sg[4 * n_pad + v2c], ay - sg[7 * n_pad + v2c]);
      const float g2 = fmaf(coef2, sg[5 * n_pad + v2c], az - sg[8 * n_pad + v2c]);
      gout[0] = p.g_tf32 ? tf32_rn(g0) : g0;
      gout[n_pad] = p.g_tf32 ? tf32_rn(g1) : g1;
      gout[2 * n_pad] = p.g_tf32 ? tf32_rn(g2) : g2;
    }
  };

  // Software pipeline over the cells of this CTA (B1/B2/B3 = split barriers, parity it & 1):
  //   wait B1 | phase A | arrive B2 | volume, arrive BV | membrane | wait B2 | hinges | wait BV |
  //   corner forces | arrive B3 | phase 0 of the NEXT cell |
  //   arrive B1 | wait B3 | phase C
  // so a warp that is early at a barrier runs ahead into work that does not depend on it.
  // Tried in round 2 and dropped (A / B on one box each, profiles/r2_ncu.md): (1) a two-barrier order with phase C of
  // cell i-1 merged into the section of phase A of cell i: 1.435 vs 1.369 ms per launch - the six corner-force gathers
  // queue in front of the vertex gathers that phase A's critical chain starts with; (2) phase C of cell i-1
  // interleaved with the hinge arithmetic of cell i (three gathers in front of each triangle's hinges, summed behind
  // them, an extra "corner forces consumed" barrier before the next stores): 1.693 vs 1.352 ms - at the 96-register
  // cap the twelve extra live registers spill, and gathers issued inside the issue-bound section wait behind it.
  if (int64_t(blockIdx.x) < p.cells) {
    phase0(0);
    bar_arrive(0);
  }
  int it = 0;
  for (int64_t cell = blockIdx.x; cell < p.cells; cell += gridDim.x, ++it) {
    const uint32_t par = uint32_t(it) & 1u;
    const float *sg = stage + (it % NSTAGE) * 12 * n_pad;
    bar_wait(0, par);                                  // B1: sx of this cell complete
    // ---- phase A: the four vertices, both normals, the volume partial ---------------------------------
    float e1[3], e2[3], f[3], n0[3], n1[3], inv0, inv1, nn0, nn1;
    float vol;
    {
      const float4 Xp = lds4(sx, lo16(qw[0])), Xq = lds4(sx, hi16(qw[0])), Xr = lds4(sx, lo16(qw[1])), Xs = lds4(sx, hi16(qw[1]));
      e1[0] = Xq.x - Xp.x; e1[1] = Xq.y - Xp.y; e1[2] = Xq.z - Xp.z;
      e2[0] = Xr.x - Xp.x; e2[1] = Xr.y - Xp.y; e2[2] = Xr.z - Xp.z;
      f[0] = Xs.x - Xp.x; f[1] = Xs.y - Xp.y; f[2] = Xs.z - Xp.z;
      // T0 = (p, q, r): N0 = e1 x e2;  T1 = (p, s, q): N1 = f x e1
      const float N0x = e1[1] * e2[2] - e1[2] * e2[1], N0y = e1[2] * e2[0] - e1[0] * e2[2], N0z = e1[0] * e2[1] - e1[1] * e2[0];
      const float N1x = f[1] * e1[2] - f[2] * e1[1], N1y = f[2] * e1[0] - f[0] * e1[2], N1z = f[0] * e1[1] - f[1] * e1[0];
      nn0 = N0x * N0x + N0y * N0y + N0z * N0z;
      nn1 = N1x * N1x + N1y * N1y + N1z * N1z;
      // 6 x signed tetrahedron volumes of both triangles (both have p as their first corner)
      vol = act ? Xp.x * (N0x + N1x) + Xp.y * (N0y + N1y) + Xp.z * (N0z + N1z) : 0.f;
      inv0 = rsqrt_fast(nn0);
      inv1 = rsqrt_fast(nn1);
      n0[0] = N0x * inv0; n0[1] = N0y * inv0; n0[2] = N0z * inv0;
      n1[0] = N1x * inv1; n1[1] = N1y * inv1; n1[2] = N1z * inv1;
      if (act) {
        sts4(sN, lo16(qw[4]), n0[0], n0[1], n0[2], inv0);
        sts4(sN, hi16(qw[4]), n1[0], n1[1], n1[2], inv1);
      }
    }
    bar_arrive(1);                                     // B2: this warp's normals are stored
    // the volume has its own barrier (BV), awaited only where the volume coefficient is used, so the
    // shuffle chain and the atomics stay off the critical path of B2
    // fixed point from here on: one REDUX instead of a shuffle tree, integer shared atomics, and the
    // result is exact, order independent and deterministic.  fx_scale leaves a factor 16 of headroom
    // over the largest per-lane partial of the rest shape; the rounding (<= 0.5 / fx_scale per lane)
    // is of the size of the fp32 rounding of the partial itself.
    {
      const int wsum = __reduce_add_sync(0xffffffffu, __float2int_rn(vol * p.fx_scale));
      if (lane == 0) {
        atomicAdd(vacc + 2 * (it & 1), wsum >> 12);          // signed high digit
        atomicAdd(vacc + 2 * (it & 1) + 1, wsum & 0xfff);    // 12-bit low digit
      }
    }
    bar_arrive(3);
    // membrane part of phase B needs this thread's registers only: it overlaps the wait for B2
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
    // the shared hinge needs this thread's own two normals only: it too runs ahead of the wait for B2
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
    bar_wait(1, par);                                  // B2: sN complete
    if (tid == 0) {
      // every thread is past phase C of the previous cell: its ring slot and the other volume
      // accumulator are free
      vacc[2 * ((it + 1) & 1)] = vacc[2 * ((it + 1) & 1) + 1] = 0;
      const int64_t nxt = cell + int64_t(NSTAGE - 1) * gridDim.x;
      if (nxt < p.cells) prefetch(nxt, (it + NSTAGE - 1) % NSTAGE);
    }
    // ---- phase B ----------------------------------------------------------------------------
    // the four neighbour normals first (independent loads in flight together), then the five hinges
    const float4 NB0 = lds4(sN, lo16(qw[2])), NB1 = lds4(sN, hi16(qw[2])), NB2 = lds4(sN, lo16(qw[3])), NB3 = lds4(sN, hi16(qw[3]));
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
    bar_wait(3, par);                                  // BV: volume accumulated
    const int2 vd = *reinterpret_cast<const int2 *>(vacc + 2 * (it & 1));
    // The int32 REDUX sums and the digit sums are exact MODULO 2^32 (a warp sum may wrap at a strongly deformed
    // iterate); the cast to int is the modular reduction that makes the difference to the rest value exact again as
    // long as |6V - 6V0| fx_scale < 2^31, i.e. while the volume stays within about +-80 % of V0 (6 V0 fx_scale is
    // 0.6 .. 1.25 x 2^31) and no lane's partial saturates the float -> int conversion (2^31: 512 x the rest-shape
    // bound).  Beyond that the volume force is garbage - the plain iteration has diverged long before, and the line
    // search takes its decisions from the fp64 objective kernel, which has no such range.  (A 64-bit conversion here
    // would be WRONG: it drops the modular reduction; tried in round 2, the violent line-search case caught it.)
    const float vc = p.vc_scale * float(int((static_cast<long long>(vd.x) << 12) + vd.y - p.fx_rest));
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
    if (act) {
      sts4(sC, lo16(qw[5]), cp[0], cp[1], cp[2], 0.f);
      sts4(sC, hi16(qw[5]), cq[0], cq[1], cq[2], 0.f);
      sts4(sC, lo16(qw[6]), cr[0], cr[1], cr[2], 0.f);
      sts4(sC, hi16(qw[6]), cs4[0], cs4[1], cs4[2], 0.f);
    }
    bar_arrive(2);
    if (cell + gridDim.x < p.cells) {                  // sx was last read in phase A (before B2)
      phase0(it + 1);
      bar_arrive(0);
    }
    bar_wait(2, par);                                  // B3: corner forces complete
    phaseC(cell, sg);
    // sN / sC are rewritten only after B1 / B2 of the next cell, which every warp reaches after this
  }
}

}  // namespace

namespace {

size_t quad_smem_bytes(const SchedDev &s, int n_pad) {
  return size_t(s.n_vslots + s.n_tslots + s.n_cslots) * 16 + size_t(NSTAGE) * 12 * n_pad * 4 + 4 * 4 + (NSTAGE + 4) * 8;
}

template <int MAXV, int MAXT, int MINB, int NPAD>
int launch_variant(const QuadParams &p, KernelCache &kc, size_t smem, int n_sm, int64_t cells, cudaStream_t s) {
  auto kernel = local_quad_kernel<MAXV, MAXT, MINB, NPAD>;
  // the opt-in attribute is per device and function, the occupancy follows from it: cached per context and type
  if (kc.quad_smem != smem) {
    if (opt_in_max_dynamic_smem(kernel) != cudaSuccess) return -1;
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, p.threads, smem) != cudaSuccess || per_sm < 1)
      return -1;
    kc.quad_smem = smem;
    kc.quad_per_sm = per_sm;
  }
  int64_t grid = int64_t(n_sm) * kc.quad_per_sm;
  if (grid > cells) grid = cells;
  kernel<<<unsigned(grid), p.threads, smem, s>>>(p);
  return 1;
}

}  // namespace

bool local_quad_supported(const TypeDev &td) {
  const SchedDev &s = td.quad;
  if (!s.valid) return false;
  if (quad_smem_bytes(s, td.n_pad) > 227 * 1024) return false;
  return s.threads <= 640 && (s.maxv == 6 || s.maxv == 8);
}

int launch_local_quad(const TypeDev &td, const BucketView &bv, int n_sm, cudaStream_t stream) {
  if (bv.cells == 0) return 0;
  if (!local_quad_supported(td)) return -1;
  const SchedDev &s = td.quad;
  QuadParams p;
  p.n = td.n; p.T = s.ttri_used; p.n_pad = td.n_pad; p.ttri = s.ttri; p.threads = s.threads; p.vstride = s.vstride;
  p.sx_bytes = s.n_vslots * 16; p.sN_bytes = s.n_tslots * 16; p.sC_bytes = s.n_cslots * 16;
  p.tri_words = s.tri_words; p.tri_consts = s.tri_consts; p.vtx_words = s.vtx_words; p.vtx_coef = s.vtx_coef;
  // fixed-point 6V as in local_sched.cu: 32 lane partials (one quad each) with 16 x headroom over the rest shape
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
  const size_t smem = quad_smem_bytes(s, td.n_pad);
  const bool v6 = s.maxv == 6;
  if (s.threads > 320) {
    if (v6 && td.n_pad == 656) return launch_variant<6, 640, 1, 656>(p, td.cache, smem, n_sm, bv.cells, stream);
    return v6 ? launch_variant<6, 640, 1, 0>(p, td.cache, smem, n_sm, bv.cells, stream)
              : launch_variant<8, 640, 1, 0>(p, td.cache, smem, n_sm, bv.cells, stream);
  }
  if (s.threads > 160)
    return v6 ? launch_variant<6, 320, 2, 0>(p, td.cache, smem, n_sm, bv.cells, stream)
              : launch_variant<8, 320, 2, 0>(p, td.cache, smem, n_sm, bv.cells, stream);
  if (v6 && td.n_pad == 176) return launch_variant<6, 160, 4, 176>(p, td.cache, smem, n_sm, bv.cells, stream);
  return v6 ? launch_variant<6, 160, 4, 0>(p, td.cache, smem, n_sm, bv.cells, stream)
            : launch_variant<8, 160, 4, 0>(p, td.cache, smem, n_sm, bv.cells, stream);
}

}  // namespace npfem
