// Local step (row a2), fp32, WARP-SPECIALISED quad path for the cell types that fill an SM with one CTA (RBC-642):
// the arithmetic of local_quad.cu (one thread per pair of adjacent triangles, quad_schedule.hpp) with the two vertex
// passes of a cell taken off the quad threads and given to a separate warp group:
//
//   quad warps   (QT = 640 threads, QREGS registers each after setmaxnreg.inc): phases A and B of cell i - gather the
//                four vertices, normals, volume, membrane, five hinges, four corner-force stores;
//   vertex warps (VT threads, VREGS registers each after setmaxnreg.dec): phase C of cell i-1 (r = coef d - b + the
//                vertex's corner forces -> global g) and phase 0 of cell i+1 (sx = x + (xl + d)), fed by the TMA ring.
//
// local_quad.cu runs these phases one after the other in the same 640 threads: its triangle sections are bound by
// instruction issue, its vertex sections by shared-memory wavefronts, and with one CTA per SM (registers) nothing
// overlaps the two.  Here they run side by side on different cells: positions are double-buffered (sx[2]), corner
// forces and normals are single-buffered behind split mbarriers that are almost never waited on, and the ring is
// split by lifetime: x, xl (dead after phase 0) in 2 stages, d, b (alive until phase C) in 4 - the same shared memory
// as the 3-stage ring of local_quad.cu, twice the prefetch distance.
//
// Barriers (mbarriers, one arrival per warp; a waiter never lags more than one phase, which is what parity waits
// can tell apart - hence the even / odd pairs where the producer can run two cells ahead):
//   VX[2]   vertex -> quad   sx[i & 1] of cell i complete                 (phase i / 2)
//   QB2     quad  -> quad    normals of cell i stored                     (phase i)
//   BV      quad  -> quad    volume of cell i accumulated                 (phase i)
//   QB3[2]  quad  -> vertex  corner forces of cell i stored; also quad -> quad: sN is free for cell i + 1
//   VC      vertex -> quad   corner forces of cell i consumed (sC free), and -> the prefetching thread: ring slot free
// Same reduced gradient r = (1 - gamma) m^ d - b + grad E(x_n + d)  (Eqs. (3)-(4), readings R5-R9),
// same fixed-point volume, bit-identical results to local_quad.cu (same operations in the same order per element).
#include "internal.h"

namespace npfem {
namespace {

constexpr int QW = 7, QK = 22;       // packed offset words / float constants per quad (quad_schedule.hpp)
constexpr int NSA = 2, NSB = 4;      // ring stages of (x, xl) and of (d, b)
#ifndef WS_VTHREADS
#define WS_VTHREADS 256          // vertex threads; the CTA owns (640 + VT) x its launch-time register count (72): setmaxnreg
#define WS_QUAD_REGS 80          // moves registers inside that pool only: 640 x QREGS + VT x VREGS <= 896 x 72 = 64,512
#define WS_VERTEX_REGS 48
#endif

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return uint32_t(__cvta_generic_to_shared(p)); }

struct WsParams {
  int n, T, n_pad, threads, vstride;   // T = quads, threads = quad threads (QT)
  int sx_bytes, sN_bytes, sC_bytes;
  const uint32_t *tri_words;   // [QW][threads]
  const float *tri_consts;     // [QK][threads]
  const uint32_t *vtx_words;   // [1 + MAXV/2][vstride]
  const float *vtx_coef;       // [vstride]
  float fx_scale;
  long long fx_rest;
  float vc_scale;
  const float *x, *xl, *d, *b; // [cells][3][n_pad]
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
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile("{\n.reg .pred q;\nmbarrier.try_wait.parity.shared::cta.b64 q, [%1], %2;\nselp.u32 %0, 1, 0, q;\n}\n"
                 : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  } while (!done);
}

// barrier indices inside `bars`: every barrier another role waits on comes as an even / odd pair (cells it & 1)
enum { B_RA = 0, B_RB = B_RA + NSA, B_VX = B_RB + NSB, B_QB2 = B_VX + 2, B_QB3 = B_QB2 + 2, B_VC = B_QB3 + 2, B_BV = B_VC + 2, B_COUNT };

template <int MAXV, int QT, int VT, int QREGS, int VREGS, int NPAD>
__global__ void __launch_bounds__(QT + VT, 1) local_ws_kernel(const WsParams p) {
  extern __shared__ __align__(16) unsigned char smem[];
  constexpr int VWORDS = 1 + MAXV / 2;
  constexpr int QWARPS = QT / 32, VWARPS = VT / 32, WORKERS = VWARPS - 1, NCH = 3;   // last vertex warp = TMA producer
  const int n = p.n, n_pad = NPAD ? NPAD : p.n_pad;
  unsigned char *sx0 = smem;                                   // [2] position buffers
  unsigned char *sN = sx0 + 2 * p.sx_bytes;
  unsigned char *sC0 = sN + p.sN_bytes;                         // [2] corner-force buffers
  float *ringA = reinterpret_cast<float *>(sC0 + 2 * p.sC_bytes);  // [NSA][x, xl][3][n_pad]
  float *ringB = ringA + NSA * 6 * n_pad;                      // [NSB][d, b][3][n_pad]
  int *vacc = reinterpret_cast<int *>(ringB + NSB * 6 * n_pad);   // [2 cells][hi, lo]
  uint64_t *bars = reinterpret_cast<uint64_t *>(vacc + 4);

  const int tid = threadIdx.x, lane = tid & 31;
  const uint32_t field_bytes = uint32_t(3 * n_pad) * 4u;

  if (tid == 0) {
    for (int s = 0; s < NSA + NSB; ++s) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(bars + s)));
    for (int s = 0; s < 2; ++s) {
      asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bars + B_VX + s)), "r"(WORKERS));
      asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bars + B_VC + s)), "r"(WORKERS));
      asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bars + B_QB2 + s)), "r"(QWARPS));
      asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bars + B_QB3 + s)), "r"(QWARPS));
    }
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bars + B_BV)), "r"(QWARPS));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    vacc[0] = vacc[1] = vacc[2] = vacc[3] = 0;
  }
  if (tid < 16) sts4(sC0 + (tid >> 3) * p.sC_bytes, uint32_t(p.sC_bytes) - 128u + 16u * (tid & 7), 0.f, 0.f, 0.f, 0.f);   // the zero slots
  __syncthreads();
  const int64_t stride = gridDim.x;
  const int64_t cnt = int64_t(blockIdx.x) < p.cells ? (p.cells - blockIdx.x + stride - 1) / stride : 0;   // this CTA's cells

  if (tid >= QT) {   // (vertex warps as the LOWEST warp ids were tried: 1.36 vs 1.27 ms, no scheduling advantage)
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(VREGS));
    const int vwarp = (tid - QT) >> 5;
    const int cnt32 = int(cnt);
    if (vwarp == WORKERS) {
      // =========================== producer: one thread keeps the two TMA rings full =============================
      if (lane != 0) return;
      auto bulk = [&](float *dst, const float *src, uint64_t *bar) {
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     ::"r"(smem_u32(dst)), "l"(src), "r"(field_bytes), "r"(smem_u32(bar)) : "memory");
      };
      auto prefetchA = [&](int k) {   // x, xl of this CTA's k-th cell -> slot k % NSA
        if (k >= cnt32) return;
        const size_t base = size_t(blockIdx.x + k * stride) * 3 * n_pad;
        const int st = k % NSA;
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bars + B_RA + st)),
                     "r"(2u * field_bytes) : "memory");
        bulk(ringA + (st * 6) * n_pad, p.x + base, bars + B_RA + st);
        bulk(ringA + (st * 6 + 3) * n_pad, p.xl + base, bars + B_RA + st);
      };
      auto prefetchB = [&](int k) {   // d, b -> slot k % NSB
        if (k >= cnt32) return;
        const size_t base = size_t(blockIdx.x + k * stride) * 3 * n_pad;
        const int st = k % NSB;
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bars + B_RB + st)),
                     "r"(2u * field_bytes) : "memory");
        bulk(ringB + (st * 6) * n_pad, p.d + base, bars + B_RB + st);
        bulk(ringB + (st * 6 + 3) * n_pad, p.b + base, bars + B_RB + st);
      };
      for (int k = 0; k < NSA; ++k) prefetchA(k);
      for (int k = 0; k < NSB; ++k) prefetchB(k);
      // in the order the events happen: phase 0 of cell it ends two cells ahead of the quads, phase C of cell it - 2
      // one cell behind them.  A slot is free once every worker is past the phase that read it last.
      for (int it = 0; it < cnt32; ++it) {
        if (it + NSA < cnt32) {
          mbar_wait(bars + B_VX + (it & 1), uint32_t(it >> 1) & 1u);
          prefetchA(it + NSA);
        }
        if (it >= 2 && it + 2 < cnt32) {
          mbar_wait(bars + B_VC + (it & 1), uint32_t((it - 2) >> 1) & 1u);
          prefetchB(it - 2 + NSB);
        }
      }
      return;
    }
    // =========================== vertex workers: phase 0 of cell it + 2, phase C of cell it ========================
    // this thread's NCH vertices (chunks vwarp, vwarp + WORKERS, ...) and their constants, in registers
    uint32_t vw[NCH][VWORDS];
    float coef[NCH];
    int vv[NCH];
#pragma unroll
    for (int j = 0; j < NCH; ++j) {
      const int v = 32 * (vwarp + WORKERS * j) + lane;
      vv[j] = v < n ? v : -1;
#pragma unroll
      for (int q = 0; q < VWORDS; ++q) vw[j][q] = v < n ? p.vtx_words[q * p.vstride + v] : 0u;
      coef[j] = v < n ? p.vtx_coef[v] : 0.f;
    }
    // phase 0 of the k-th cell: sx[k & 1][slot(v)] = (x + (xl + d), 0), the current position from the two-float x_n
    auto phase0 = [&](int k) {
      const int sa_i = k % NSA, sb_i = k % NSB;
      mbar_wait(bars + B_RA + sa_i, uint32_t(k / NSA) & 1u);
      mbar_wait(bars + B_RB + sb_i, uint32_t(k / NSB) & 1u);
      const float *sa = ringA + sa_i * 6 * n_pad, *sb = ringB + sb_i * 6 * n_pad;
      unsigned char *sx = sx0 + (k & 1) * p.sx_bytes;
#pragma unroll
      for (int j = 0; j < NCH; ++j) {
        const int v = vv[j];
        if (v >= 0)
          sts4(sx, vw[j][0] & 0xffffu, sa[v] + (sa[3 * n_pad + v] + sb[v]), sa[n_pad + v] + (sa[4 * n_pad + v] + sb[n_pad + v]),
               sa[2 * n_pad + v] + (sa[5 * n_pad + v] + sb[2 * n_pad + v]), 0.f);
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(bars + B_VX + (k & 1));
    };
    if (cnt32 > 0) phase0(0);
    if (cnt32 > 1) phase0(1);
    for (int it = 0; it < cnt32; ++it) {
      const uint32_t par = uint32_t(it) & 1u, ph = uint32_t(it >> 1) & 1u;
      if (it + 2 < cnt32) {
        mbar_wait(bars + B_QB2 + par, ph);       // every quad warp has gathered cell it's positions: sx[par] is free
        phase0(it + 2);
      }
      mbar_wait(bars + B_QB3 + par, ph);         // corner forces of cell `it` stored
      // ---- phase C: r = coef d - b + sum of the vertex's corner forces -> global ----------------------------
      const float *sb = ringB + (it % NSB) * 6 * n_pad;
      const unsigned char *sC = sC0 + par * p.sC_bytes;
      float *gcell = p.g + size_t(blockIdx.x + it * stride) * 3 * n_pad;
#pragma unroll
      for (int j = 0; j < NCH; ++j) {
        const int v = vv[j];
        if (v >= 0) {
          // all gathers in flight together; the sums run in slot order 0 .. MAXV-1 like local_quad.cu (bit-identical)
          float4 f[MAXV];
#pragma unroll
          for (int q = 0; q < MAXV; q += 2) {
            const uint32_t w = vw[j][1 + (q >> 1)];
            f[q] = lds4(sC, w & 0xffffu);
            f[q + 1] = lds4(sC, w >> 16);
          }
          float ax = 0.f, ay = 0.f, az = 0.f;
#pragma unroll
          for (int q = 0; q < MAXV; ++q) { ax += f[q].x; ay += f[q].y; az += f[q].z; }
          float g0 = fmaf(coef[j], sb[v], ax - sb[3 * n_pad + v]);
          float g1 = fmaf(coef[j], sb[n_pad + v], ay - sb[4 * n_pad + v]);
          float g2 = fmaf(coef[j], sb[2 * n_pad + v], az - sb[5 * n_pad + v]);
          if (p.g_tf32) { g0 = tf32_rn(g0); g1 = tf32_rn(g1); g2 = tf32_rn(g2); }
          gcell[v] = g0;
          gcell[n_pad + v] = g1;
          gcell[2 * n_pad + v] = g2;
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(bars + B_VC + par);
    }
    return;
  }

  // =========================== quad warps: phases A and B of cell `it` ===========================================
  asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(QREGS));
  // qw: 0 = p | q, 1 = r | s (vertex slots), 2 = n0 | n1 (normals across q-r, r-p), 3 = n2 | n3 (across p-s, s-q),
  //     4 = own normal slots T0 | T1, 5 = corner slots p | q, 6 = r | s          (16-bit byte offsets)
  // qk: 0..5 = R11 R12 R22 J tA tC of T0 = (p, q, r), 6..11 = of T1 = (p, s, q), 12..16 = k_b cos theta0 and
  //     17..21 = k_b sin theta0 of the hinges  shared p-q, q-r, r-p, p-s, s-q
  uint32_t qw[QW];
  float qk[QK];
  const int qtid = tid;
  const bool act = qtid < p.T;
#pragma unroll
  for (int q = 0; q < QW; ++q) qw[q] = p.tri_words[q * QT + qtid];
#pragma unroll
  for (int q = 0; q < QK; ++q) qk[q] = p.tri_consts[q * QT + qtid];
  auto arrive = [&](int which) {
    __syncwarp();
    if (lane == 0) mbar_arrive(bars + which);
  };
  for (int64_t it64 = 0; it64 < cnt; ++it64) {
    const int it = int(it64);
    const uint32_t par = uint32_t(it) & 1u;
    const unsigned char *sx = sx0 + par * p.sx_bytes;
    unsigned char *sC = sC0 + par * p.sC_bytes;
    mbar_wait(bars + B_VX + par, uint32_t(it >> 1) & 1u);   // VX: sx[par] of this cell complete
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
      // sN is free once every quad warp has stored its corner forces of the previous cell (its hinges are done)
      if (it > 0) mbar_wait(bars + B_QB3 + ((it - 1) & 1), uint32_t((it - 1) >> 1) & 1u);
      if (act) {
        sts4(sN, lo16(qw[4]), n0[0], n0[1], n0[2], inv0);
        sts4(sN, hi16(qw[4]), n1[0], n1[1], n1[2], inv1);
      }
    }
    arrive(B_QB2 + int(par));                          // QB2: this warp's normals are stored (its sx gathers are done)
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
    arrive(B_BV);
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
    mbar_wait(bars + B_QB2 + par, uint32_t(it >> 1) & 1u);   // QB2: sN complete
    // every quad warp is past its read of the previous cell's volume: the other accumulator is free
    if (qtid == 0) vacc[2 * ((it + 1) & 1)] = vacc[2 * ((it + 1) & 1) + 1] = 0;
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
    mbar_wait(bars + B_BV, par);                       // BV: volume accumulated
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
    if (it > 1) mbar_wait(bars + B_VC + par, uint32_t((it - 2) >> 1) & 1u);   // sC[par] of cell it - 2 consumed
    if (act) {
      sts4(sC, lo16(qw[5]), cp[0], cp[1], cp[2], 0.f);
      sts4(sC, hi16(qw[5]), cq[0], cq[1], cq[2], 0.f);
      sts4(sC, lo16(qw[6]), cr[0], cr[1], cr[2], 0.f);
      sts4(sC, hi16(qw[6]), cs4[0], cs4[1], cs4[2], 0.f);
    }
    arrive(B_QB3 + int(par));                          // QB3: this warp's corner forces are stored
  }
}

}  // namespace

namespace {

constexpr int WS_QT = 640, WS_VT = WS_VTHREADS, WS_QREGS = WS_QUAD_REGS, WS_VREGS = WS_VERTEX_REGS;

size_t ws_smem_bytes(const SchedDev &s, int n_pad) {
  return size_t(2 * s.n_vslots + s.n_tslots + 2 * s.n_cslots) * 16 + size_t(NSA + NSB) * 6 * n_pad * 4 +
         4 * 4 + B_COUNT * 8;
}

template <int MAXV, int NPAD>
int launch_variant(const WsParams &p, KernelCache &kc, size_t smem, int n_sm, int64_t cells, cudaStream_t s) {
  auto kernel = local_ws_kernel<MAXV, WS_QT, WS_VT, WS_QREGS, WS_VREGS, NPAD>;
  if (kc.ws_smem != smem) {
    if (opt_in_max_dynamic_smem(kernel) != cudaSuccess) return -1;
    kc.ws_smem = smem;
  }
  const int64_t grid = cells < n_sm ? cells : n_sm;     // one CTA per SM: it holds all 64 K registers
  kernel<<<unsigned(grid), WS_QT + WS_VT, smem, s>>>(p);
  return 1;
}

}  // namespace

bool local_ws_supported(const TypeDev &td) {
  const SchedDev &s = td.quad;
  if (!s.valid || s.threads != WS_QT || (s.maxv != 6 && s.maxv != 8)) return false;
  return ws_smem_bytes(s, td.n_pad) <= 227 * 1024;
}

int launch_local_ws(const TypeDev &td, const BucketView &bv, int n_sm, cudaStream_t stream) {
  if (bv.cells == 0) return 0;
  if (!local_ws_supported(td)) return -1;
  const SchedDev &s = td.quad;
  WsParams p;
  p.n = td.n; p.T = s.ttri_used; p.n_pad = td.n_pad; p.threads = s.threads; p.vstride = s.vstride;
  p.sx_bytes = s.n_vslots * 16; p.sN_bytes = s.n_tslots * 16; p.sC_bytes = s.n_cslots * 16;
  p.tri_words = s.tri_words; p.tri_consts = s.tri_consts; p.vtx_words = s.vtx_words; p.vtx_coef = s.vtx_coef;
  // fixed-point 6V as in local_quad.cu: 32 lane partials (one quad each) with 16 x headroom over the rest shape
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
  const size_t smem = ws_smem_bytes(s, td.n_pad);
  if (s.maxv == 6) {
    if (td.n_pad == 656) return launch_variant<6, 656>(p, td.cache, smem, n_sm, bv.cells, stream);
    return launch_variant<6, 0>(p, td.cache, smem, n_sm, bv.cells, stream);
  }
  return launch_variant<8, 0>(p, td.cache, smem, n_sm, bv.cells, stream);
}

}  // namespace npfem
