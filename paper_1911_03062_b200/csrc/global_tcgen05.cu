// Global step (row a3) on the 5th-generation tensor cores: d <- d - g H~^-1 for a whole type
// bucket as ONE TF32 GEMM  D[3*cells x n_pad] -= G[3*cells x n_pad] . W[n_pad x n_pad]
// (Eq. (4), reading R1; x in R^{n x 3}, matrices n x n).
//
// Cells of one type share the rest shape, hence the operator: the structure is a dense
// contraction of one constant matrix against many right-hand sides, which is the only place of
// the path where tensor cores apply.  Increment form keeps TF32 safe: the rounding lands on the
// small update g W, not on d.
//
// Kernel: persistent, one CTA per SM in clusters of CL = 2, warp-specialised.
//   warp 0   TMA producer : own G tile [128 x 32 fp32] + this CTA's 1/CL of the W tile [N_pass x 32],
//                           multicast to every CTA of the cluster, per K chunk; 128B swizzle; ring of up to
//                           4 stages sized per launch
//   warp 1   MMA issuer   : tcgen05.mma.cta_group::1.kind::tf32, M = 128, N = N_pass <= 256, two accumulators
//                           in the 512 TMEM columns; A negated in the instruction descriptor (acc = -G W);
//                           its commit frees the ring slot in every CTA of the cluster
//   warps 2-5 epilogue    : [32 x 32] tiles: TMA load of d into swizzled shared memory -> tcgen05.ld ->
//                           d_scale d + acc in place (row per lane, conflict-free) -> TMA store
// Work item of a cluster = (CL consecutive M tiles, N pass); the passes of one group are adjacent items
// (neighbouring clusters at about the same time), so the repeated G reads are L2 hits.
// Split-operator mode (k_segs = 2, NPFEM_OPT_GLOBAL_STEP_MATH = 2): [g g] . [W_hi; W_lo], the operator to ~fp32 accuracy
// (the reduced-gradient identity is exact only for the exact H~^-1; TF32 rounding of W biases the
// fixed point).  Line-search mode (k_segs = 3): the 3xTF32 product [g_hi g_lo g_hi] . [W_hi; W_hi; W_lo] as one GEMM with K = 3 n_pad;
// the producer switches tensor maps per K segment, nothing else changes.
#include <cuda.h>

#include "internal.h"

namespace npfem {
namespace {

constexpr int BM = 128;          // rows per tile (TMEM lanes)
constexpr int BK = 32;           // fp32 per K chunk = 128 bytes = one swizzle row
constexpr int UMMA_K = 8;        // K per tcgen05.mma for tf32 (32 bytes)
constexpr int MAX_STAGES = 4;      // ring depth is chosen per launch: as many stages as fit next to the epilogue tiles
constexpr int CL = 2;             // thread-block cluster: CL CTAs work on CL consecutive M tiles and share every W tile
constexpr int MAX_NPASS = 256;   // accumulator columns per pass: two accumulators fit the 512 TMEM columns
constexpr int A_BYTES = BM * BK * 4;
constexpr int B_BYTES = MAX_NPASS * BK * 4;
constexpr int EBUF = 3;           // per epilogue warp: ring of [32 rows x 32 cols] fp32 staging tiles (4 KB each)
constexpr int EPI_BYTES = 4 * EBUF * 4096;
constexpr int SMEM_LIMIT = 227 * 1024;

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return uint32_t(__cvta_generic_to_shared(p)); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  } while (!done);
}

__device__ __forceinline__ void tma_load_2d(void *smem_dst, const CUtensorMap *map, int x, int y, uint64_t *bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
      ::"r"(smem_u32(smem_dst)), "l"(map), "r"(smem_u32(bar)), "r"(x), "r"(y) : "memory");
}

// same, delivered to the same shared-memory offset of every CTA in `mask` (their full barriers at the
// same offset receive the complete_tx)
__device__ __forceinline__ void tma_load_2d_mc(void *smem_dst, const CUtensorMap *map, int x, int y, uint64_t *bar,
                                               uint16_t mask) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster [%0], [%1, {%3, %4}], [%2], %5;"
      ::"r"(smem_u32(smem_dst)), "l"(map), "r"(smem_u32(bar)), "r"(x), "r"(y), "h"(mask) : "memory");
}
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

__device__ __forceinline__ void tma_store_2d(const CUtensorMap *map, int x, int y, const void *smem_src) {
  asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%2, %3}], [%1];"
               ::"l"(map), "r"(smem_u32(smem_src)), "r"(x), "r"(y) : "memory");
}

// K-major, 128B-swizzled operand tile: 8-row atoms of 1024 bytes (SBO), version 1 (sm_100)
__device__ __forceinline__ uint64_t make_smem_desc(uint32_t saddr) {
  uint64_t desc = 0;
  desc |= uint64_t((saddr & 0x3FFFF) >> 4);          // start address, bits [0,14)
  desc |= uint64_t(1) << 16;                         // leading byte offset (unused for swizzled K-major)
  desc |= uint64_t(1024 >> 4) << 32;                 // stride byte offset, bits [32,46)
  desc |= uint64_t(1) << 46;                         // descriptor version for Blackwell
  desc |= uint64_t(2) << 61;                         // SWIZZLE_128B
  return desc;
}

// kind::tf32, fp32 accumulate, A and B K-major, A negated
__host__ __device__ constexpr uint32_t make_idesc(int M, int N) {
  return (1u << 4) | (2u << 7) | (2u << 10) | (1u << 13) | (uint32_t(N >> 3) << 17) | (uint32_t(M >> 4) << 24);
}

__device__ __forceinline__ void umma_tf32(uint32_t tmem_d, uint64_t a_desc, uint64_t b_desc, uint32_t idesc,
                                          uint32_t accumulate) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "setp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n"
      "}\n" ::"r"(tmem_d), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t *bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar))
               : "memory");
}

// arrives on the barrier at this offset in every CTA of `mask` once the MMAs issued so far have retired
__device__ __forceinline__ void umma_commit_mc(uint64_t *bar, uint16_t mask) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
               ::"r"(smem_u32(bar)), "h"(mask) : "memory");
}

struct GemmParams {
  float *D;            // [rows][n_pad], updated in place
  int64_t rows;
  int n_pad;
  int n_pass;          // accumulator columns per pass = N of the MMA (multiple of 16, <= MAX_NPASS)
  int passes;          // ceil(n_pad / n_pass)
  int k_chunks;        // ceil(n_pad / BK)
  int k_segs;          // 1; 2: [g g] . [W_hi; W_lo]; 3: K-concatenated 3xTF32 product [g_hi g_lo g_hi] . [W_hi; W_hi; W_lo]
  int seg_g2, seg_w2;  // bit s set: K segment s reads the second G map (g_lo) / the second W map (W_lo)
  int64_t m_tiles;
  float d_scale;       // d <- d_scale * d + acc
  int stages;          // depth of the operand ring (<= MAX_STAGES)
  int stage_bytes;     // A tile + W tile of n_pass rows, multiple of 1024
};

__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&r)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
        "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr));
}

__global__ void __launch_bounds__(192, 1)
global_tcgen05_kernel(const __grid_constant__ CUtensorMap map_g, const __grid_constant__ CUtensorMap map_w,
                      const __grid_constant__ CUtensorMap map_d, const __grid_constant__ CUtensorMap map_g2,
                      const __grid_constant__ CUtensorMap map_w2, const GemmParams p) {
  extern __shared__ unsigned char smem_raw[];
  __shared__ uint64_t full_bar[MAX_STAGES], empty_bar[MAX_STAGES], tmem_full_bar[2], tmem_empty_bar[2], epi_full[4 * EBUF];
  __shared__ uint32_t tmem_base_sh;
  unsigned char *smem = reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  // work item of a CLUSTER = (group of CL consecutive M tiles, N pass); CTA `rank` takes tile CL*group + rank.
  // A tile past the end is processed like any other (TMA zero-fills, the epilogue stores nothing) so
  // that both CTAs keep the multicast protocol in step.
  const uint32_t rank = cluster_ctarank();
  const int64_t n_items = ((p.m_tiles + CL - 1) / CL) * p.passes;
  const int64_t first_item = blockIdx.x / CL, item_step = gridDim.x / CL;
  constexpr uint16_t MASK = uint16_t((1u << CL) - 1u);

  if (threadIdx.x == 0) {
    for (int s = 0; s < p.stages; ++s) {
      mbar_init(&full_bar[s], 1);
      mbar_init(&empty_bar[s], CL);                         // every CTA of the cluster reads what lands here
    }
    for (int a = 0; a < 2; ++a) {
      mbar_init(&tmem_full_bar[a], 1);
      mbar_init(&tmem_empty_bar[a], 128);
    }
    for (int b = 0; b < 4 * EBUF; ++b) mbar_init(&epi_full[b], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) {   // TMEM: all 512 columns (one CTA per SM) = two accumulators of <= 256 columns
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(&tmem_base_sh)));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  cluster_sync_all();                                       // the peers' barriers exist before anyone signals them
  asm volatile("tcgen05.fence::after_thread_sync;");
  const uint32_t tmem_base = tmem_base_sh;

  if (warp == 0) {
    // ===== TMA producer =====
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0;
      const uint32_t tx = A_BYTES + uint32_t(p.n_pass) * BK * 4;
      const int w_rows = p.n_pass / CL;                     // this CTA's slice of the W tile (multiple of 8 rows)
      for (int64_t item = first_item; item < n_items; item += item_step) {
        const int row0 = int(((item / p.passes) * CL + rank) * BM), col0 = int(item % p.passes) * p.n_pass;
        for (int seg = 0; seg < p.k_segs; ++seg) {
          const CUtensorMap *mg = (p.seg_g2 >> seg) & 1 ? &map_g2 : &map_g, *mw = (p.seg_w2 >> seg) & 1 ? &map_w2 : &map_w;
          for (int kc = 0; kc < p.k_chunks; ++kc) {
            mbar_wait(&empty_bar[stage], phase ^ 1);        // this slot is free in EVERY CTA of the cluster
            unsigned char *sa = smem + stage * p.stage_bytes, *sb = sa + A_BYTES;
            mbar_expect_tx(&full_bar[stage], tx);           // own G tile + all CL slices of the W tile
            tma_load_2d(sa, mg, kc * BK, row0, &full_bar[stage]);
            tma_load_2d_mc(sb + size_t(rank) * w_rows * BK * 4, mw, kc * BK, col0 + int(rank) * w_rows,
                           &full_bar[stage], MASK);
            if (++stage == p.stages) { stage = 0; phase ^= 1; }
          }
        }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer =====
    if (lane == 0) {
      int stage = 0;
      uint32_t phase = 0, li = 0;
      const uint32_t idesc = make_idesc(BM, p.n_pass);
      for (int64_t item = first_item; item < n_items; item += item_step, ++li) {
        const uint32_t acc = li & 1u, acc_phase = (li >> 1) & 1u;
        mbar_wait(&tmem_empty_bar[acc], acc_phase ^ 1);     // epilogue has drained this accumulator
        asm volatile("tcgen05.fence::after_thread_sync;");
        const uint32_t tacc = tmem_base + acc * MAX_NPASS;
        for (int kc = 0; kc < p.k_chunks * p.k_segs; ++kc) {
          mbar_wait(&full_bar[stage], phase);
          asm volatile("tcgen05.fence::after_thread_sync;");
          const uint32_t sa = smem_u32(smem + stage * p.stage_bytes), sb = sa + A_BYTES;
#pragma unroll
          for (int k = 0; k < BK / UMMA_K; ++k)
            umma_tf32(tacc, make_smem_desc(sa + k * UMMA_K * 4), make_smem_desc(sb + k * UMMA_K * 4), idesc,
                      (kc | k) != 0);
          umma_commit_mc(&empty_bar[stage], MASK);          // frees the slot in every CTA when these MMAs retire
          if (++stage == p.stages) { stage = 0; phase ^= 1; }
        }
        umma_commit(&tmem_full_bar[acc]);                   // accumulator complete
      }
    }
  } else {
    // ===== epilogue: warps 2..5 own TMEM lanes 32*(warp%4) .. +31; overlaps the next item's MMAs =====
    // d <- d_scale d + acc in tiles of [32 rows x 32 columns], each warp on its own ring of
    // EBUF staging tiles: TMA load (128B swizzle) -> every lane updates ITS row in shared memory
    // (conflict-free thanks to the swizzle) -> TMA store.  All global traffic of the epilogue is
    // full 128-byte rows moved by the TMA unit; a row-per-lane LDG/STG pattern (32 lines per warp
    // instruction) held the previous version to a third of the tensor peak.
    const int lane_base = (warp & 3) * 32;
    unsigned char *ebuf = smem + p.stages * p.stage_bytes + (warp & 3) * (EBUF * 4096);
    uint64_t *efull = &epi_full[(warp & 3) * EBUF];
    const int n_chunks = (p.n_pass + 31) / 32;
    uint32_t g = 0;                                         // tiles this warp has processed (ring position)
    uint32_t li = 0;
    for (int64_t item = first_item; item < n_items; item += item_step, ++li) {
      const uint32_t acc = li & 1u, acc_phase = (li >> 1) & 1u;
      const int row0w = int(((item / p.passes) * CL + rank) * BM) + lane_base;
      const int col0 = int(item % p.passes) * p.n_pass;
      const uint32_t tacc = tmem_base + acc * MAX_NPASS + (uint32_t(lane_base) << 16);
      auto issue_load = [&](int c, uint32_t gc) {           // lane 0 only
        const uint32_t b = gc % EBUF;
        asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");   // the store that last read this tile is done
        mbar_expect_tx(&efull[b], 4096);
        tma_load_2d(ebuf + b * 4096, &map_d, col0 + 32 * c, row0w, &efull[b]);
      };
      if (lane == 0) issue_load(0, g);                      // requested before the accumulator is awaited
      mbar_wait(&tmem_full_bar[acc], acc_phase);
      asm volatile("tcgen05.fence::after_thread_sync;");
      for (int c = 0; c < n_chunks; ++c) {
        const uint32_t gc = g + uint32_t(c), b = gc % EBUF;
        if (lane == 0 && c + 1 < n_chunks) issue_load(c + 1, gc + 1);   // tile gc-2's store may still run
        uint32_t r[32];
        {
          uint32_t r0[16], r1[16];
          tmem_ld16(tacc + uint32_t(32 * c), r0);
          tmem_ld16(tacc + uint32_t(32 * c) + 16u, r1);     // may read an unused column block: clipped by the store
          asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
          for (int q = 0; q < 16; ++q) { r[q] = r0[q]; r[16 + q] = r1[q]; }
        }
        mbar_wait(&efull[b], (gc / EBUF) & 1u);
        float4 *rowp = reinterpret_cast<float4 *>(ebuf + b * 4096 + lane * 128);
#pragma unroll
        for (int q = 0; q < 8; ++q) {
          float4 *slot = rowp + (q ^ (lane & 7));           // 128B swizzle: 16-byte chunk q of row r sits at q ^ (r % 8)
          float4 v = *slot;
          v.x = fmaf(p.d_scale, v.x, __uint_as_float(r[4 * q]));
          v.y = fmaf(p.d_scale, v.y, __uint_as_float(r[4 * q + 1]));
          v.z = fmaf(p.d_scale, v.z, __uint_as_float(r[4 * q + 2]));
          v.w = fmaf(p.d_scale, v.w, __uint_as_float(r[4 * q + 3]));
          *slot = v;
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncwarp();
        if (lane == 0) {                                    // rows / columns past the matrix are clipped by the TMA unit
          tma_store_2d(&map_d, col0 + 32 * c, row0w, ebuf + b * 4096);
          asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
      }
      g += uint32_t(n_chunks);
      asm volatile("tcgen05.fence::before_thread_sync;");
      mbar_arrive(&tmem_empty_bar[acc]);
    }
    if (lane == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
  }
  __syncthreads();
  cluster_sync_all();                                       // no CTA leaves while a peer may still signal it
  if (warp == 1) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem_base));
  }
}

// ---- host: tensor maps --------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void *p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  }
  return fn;
}

// 2-D fp32 row-major tensor [rows][cols] (cols contiguous, row pitch `pitch` elements), box [box_rows][32]
bool make_map(CUtensorMap *map, const void *base, uint64_t rows, uint64_t cols, uint64_t pitch, uint32_t box_rows) {
  EncodeTiledFn enc = get_encode();
  if (!enc) return false;
  const cuuint64_t dims[2] = {cols, rows};
  const cuuint64_t strides[1] = {pitch * sizeof(float)};
  const cuuint32_t box[2] = {BK, box_rows};
  const cuuint32_t estr[2] = {1, 1};
  return enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void *>(base), dims, strides, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace

// shape of the tensor-core path for a type: false when unsupported (caller uses the SIMT GEMM)
static bool gemm_shape(const TypeDev &td, GemmParams &p) {
  p.n_pad = td.n_pad;
  p.passes = (td.n_pad + MAX_NPASS - 1) / MAX_NPASS;
  // the epilogue moves 32-column tiles: with several passes a pass must END on a tile boundary, or its
  // last tile would also rewrite the first columns of the next pass (one pass: the TMA store clips at n_pad)
  const int gran = p.passes > 1 ? 32 : 16;
  p.n_pass = ((td.n_pad + p.passes - 1) / p.passes + gran - 1) / gran * gran;
  if (p.n_pass > MAX_NPASS || p.n_pass < 16 || (p.n_pass / CL) % 8 != 0 || td.Hinv == nullptr) return false;
  p.k_chunks = (td.n_pad + BK - 1) / BK;
  p.stage_bytes = A_BYTES + (p.n_pass * BK * 4 + 1023) / 1024 * 1024;
  p.stages = (SMEM_LIMIT - 1024 - EPI_BYTES) / p.stage_bytes;
  if (p.stages > MAX_STAGES) p.stages = MAX_STAGES;
  return p.stages >= 2;
}

bool global_tcgen05_supported(const TypeDev &td) {
  GemmParams p{};
  return gemm_shape(td, p) && get_encode() != nullptr;
}

// d <- d_scale d - g Hinv.  Returns #launches, -1 if the shape is unsupported (npfem_step decides BEFORE launching
// which GEMM a bucket takes: global_tcgen05_supported), -2 if the launch itself failed (an NPFEM_ECUDA for the
// caller, never a silent fall back to the SIMT GEMM).
// w_lo alone: d <- d_scale d - (g W + g W_lo) (split operator).  g_lo and w_lo: the line search's 3xTF32 product d <- d_scale d - (g W + g_lo W + g W_lo) as ONE
// GEMM with the three products concatenated along K (g = bv.field[F_G] holds the TF32 high part, W = Hinv_tf32).
int launch_global_tcgen05(const TypeDev &td, const BucketView &bv, int n_sm, double d_scale,
                          cudaStream_t s, const void *g_lo, const void *w_lo) {
  if (bv.cells == 0) return 0;
  GemmParams p{};
  if (!gemm_shape(td, p)) return -1;
  p.D = static_cast<float *>(bv.field[F_D]);
  p.rows = bv.cells * 3;
  p.m_tiles = (p.rows + BM - 1) / BM;
  p.d_scale = float(d_scale);
  CUtensorMap map_g, map_w, map_d;
  if (!make_map(&map_g, bv.field[F_G], uint64_t(p.rows), uint64_t(td.n_pad), uint64_t(td.n_pad), BM)) return -2;
  if (!make_map(&map_w, td.Hinv_tf32 ? td.Hinv_tf32 : td.Hinv, uint64_t(td.n_pad), uint64_t(td.n_pad), uint64_t(td.n_pad), uint32_t(p.n_pass / CL)))
    return -2;
  CUtensorMap map_g2 = map_g, map_w2 = map_w;
  p.k_segs = 1;
  p.seg_g2 = p.seg_w2 = 0;
  if (w_lo) {
    if (!make_map(&map_w2, w_lo, uint64_t(td.n_pad), uint64_t(td.n_pad), uint64_t(td.n_pad), uint32_t(p.n_pass / CL))) return -2;
    if (g_lo) {          // (g_hi, W_hi), (g_lo, W_hi), (g_hi, W_lo)
      if (!make_map(&map_g2, g_lo, uint64_t(p.rows), uint64_t(td.n_pad), uint64_t(td.n_pad), BM)) return -2;
      p.k_segs = 3;
      p.seg_g2 = 0b010;
      p.seg_w2 = 0b100;
    } else {             // (g, W_hi), (g, W_lo)
      p.k_segs = 2;
      p.seg_w2 = 0b010;
    }
  }
  // epilogue tiles: [32 rows][32 columns] of D (in-place update)
  if (!make_map(&map_d, bv.field[F_D], uint64_t(p.rows), uint64_t(td.n_pad), uint64_t(td.n_pad), 32))
    return -2;
  const int smem_bytes = p.stages * p.stage_bytes + EPI_BYTES + 1024;
  if (td.cache.tc_smem == 0) {   // per context and type: the attribute is per device (always the architectural maximum)
    if (opt_in_max_dynamic_smem(global_tcgen05_kernel) != cudaSuccess) return -2;
    td.cache.tc_smem = smem_bytes;
  }
  // the passes of one group of M tiles are adjacent items: they run on neighbouring clusters at about
  // the same time, so the repeated reads of the G tiles are L2 hits
  const int64_t items = ((p.m_tiles + CL - 1) / CL) * p.passes;
  const int64_t clusters = items < n_sm / CL ? items : n_sm / CL;
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(unsigned(clusters * CL));
  cfg.blockDim = dim3(192);
  cfg.dynamicSmemBytes = size_t(smem_bytes);
  cfg.stream = s;
  cudaLaunchAttribute attrs[1];
  attrs[0].id = cudaLaunchAttributeClusterDimension;
  attrs[0].val.clusterDim.x = CL;
  attrs[0].val.clusterDim.y = 1;
  attrs[0].val.clusterDim.z = 1;
  cfg.attrs = attrs;
  cfg.numAttrs = 1;
  if (cudaLaunchKernelEx(&cfg, global_tcgen05_kernel, map_g, map_w, map_d, map_g2, map_w2, p) != cudaSuccess) return -2;
  return 1;
}

}  // namespace npfem
