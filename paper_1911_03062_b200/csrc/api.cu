// C ABI of libnpfem_b200.so (include/npfem.h): context, workspace layout, call orchestration.
// Every arithmetic step of the path runs in the CUDA kernels of this directory; there is no
// CPU fallback.
#include <algorithm>
#include <chrono>
#include <cstdio>
#include <cstring>
#include <new>

#include "internal.h"
#include "local_schedule.hpp"
#include "quad_schedule.hpp"
#include "quadmp_schedule.hpp"

static_assert(npfem::QMP_MAX_PASSES == 4 && npfem::QMP_THREADS == 640,
              "local_quadmp.cu (NP, TH) and QuadMpDev::list_len are written for 4 passes of 640 quads");

using namespace npfem;

struct npfem_ctx {
  int precision = NPFEM_F32, device = 0, n_sm = 148;
  cudaStream_t stream = nullptr;
  double dt = 0;
  int64_t n_cells = 0, total_vertices = 0;
  std::vector<HostTypeData> host_types;
  std::vector<LocalSchedule> sched;       // fp32 contexts: scheduled local step, per type (may be invalid)
  std::vector<QuadSchedule> quad;         // fp32 contexts: quad local step, per type (may be invalid)
  std::vector<QuadMpSchedule> quadmp;     // fp32 contexts: multi-pass quad local step of larger meshes (may be invalid)
  std::vector<TypeDev> types;
  std::vector<Bucket> buckets;            // one per type
  std::vector<BucketView> views;
  std::vector<int32_t> type_of_cell, slot_of_cell;
  std::vector<int64_t> user_offset_all;   // [n_cells+1] element offsets in all-cells order
  std::vector<uint8_t> cell_is_set;
  std::vector<uint32_t> seen_epoch;       // duplicate detection in id lists
  uint32_t epoch = 0;
  int64_t n_set = 0;
  // workspace
  unsigned char *ws = nullptr;
  size_t ws_bytes = 0;
  bool ws_owned = false, ready = false;
  struct Layout {
    std::vector<size_t> type_off[28];     // per type: tri, nbr, rest, hinge, corner, vnbr, w, mass, inv_area, Hinv, Hinv_tf32
    std::vector<size_t> field_off[F_COUNT], origin_off, cellid_off, scratch_off;
    size_t views_off = 0, refs_all_off = 0, refs_tmp_off = 0, stage_a_off = 0, stage_b_off = 0, stage_c_off = 0, total = 0;
    // create-time arena (the fp64 H~, its inverse and the Newton-Schulz temporaries of ONE type at a time): starts
    // right after the per-type tables and is overlaid by the state fields, which are first written by set_state
    size_t setup_off = 0, setup_bytes = 0;
  } lay;
  // Optional features (diagnostics history, line-search state and operands, collision tables) live in a SCRATCH
  // arena: bound by the caller (npfem_bind_scratch) or, when the library owns its workspace, allocated by the call
  // that enables the feature - never inside npfem_step.
  struct FeatureMem { unsigned char *base = nullptr; size_t bytes = 0; bool owned = false, wanted = false, live = false; };
  FeatureMem feat[3];                     // index = log2(NPFEM_FEATURE_*)
  BucketView *views_dev = nullptr;
  CellRef *refs_all_dev = nullptr, *refs_tmp_dev = nullptr;
  std::vector<int64_t *> cell_id_dev;
  void *stage_a = nullptr, *stage_b = nullptr, *stage_c = nullptr;
  // npfem_step_host: copy streams and per-chunk events, created on first use
  cudaStream_t h2d_stream = nullptr, d2h_stream = nullptr;
  std::vector<cudaEvent_t> io_events;
  // diagnostics
  bool diagnostics = false;
  double *history_dev = nullptr;          // [NPFEM_MAX_ITERATIONS + 1][n_cells], in feat[0]
  int history_entries = 0;
  int64_t opt_global_math = 0, opt_local_impl = 0, opt_fused_step = 0;
  // line search (npfem_set_line_search)
  int ls_max_halvings = 0;
  double ls_c1 = 1e-4, ls_tol = 0.0;
  std::vector<LineSearchDev> ls;          // per bucket, carved from feat[1]
  bool ls_ran = false;
  // coupling-side options
  bool median_filter = false;
  double v_max = 0.0;
  std::vector<CollisionDev> col;          // per bucket, carved from feat[2]
  CollisionDev *col_dev = nullptr;        // the same table on the device
  bool col_active = false;
  int64_t launches = 0;
  // kernel timing (NPFEM_OPT_KERNEL_TIMING)
  bool timing = false;
  struct TimedSpan { cudaEvent_t a, b; int kind, type; int launches; };
  std::vector<TimedSpan> spans;
  std::vector<cudaEvent_t> event_pool;
  std::vector<double> kind_ms;
  std::vector<int64_t> kind_launches;
  bool sticky = false;
  std::string err;
};

namespace {

thread_local std::string g_create_error;

size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }
size_t esize(int precision) { return precision == NPFEM_F32 ? 4 : 8; }

int fail(npfem_ctx *c, int code, const std::string &msg) {
  if (c) {
    c->err = msg;
    if (code == NPFEM_ECUDA) c->sticky = true;
  } else {
    g_create_error = msg;
  }
  return code;
}

#define NPFEM_CUDA(c, call)                                                              \
  do {                                                                                   \
    cudaError_t e_ = (call);                                                             \
    if (e_ != cudaSuccess)                                                               \
      return fail((c), NPFEM_ECUDA, std::string(#call ": ") + cudaGetErrorString(e_));   \
  } while (0)

int check_launch(npfem_ctx *c, int n, const char *what) {
  if (n == -2) {   // the launch (or its setup: attribute, tensor map) failed: a CUDA error, sticky
    const cudaError_t e = cudaGetLastError();
    return fail(c, NPFEM_ECUDA, std::string(what) + ": launch failed: " + (e != cudaSuccess ? cudaGetErrorString(e) : "driver call refused"));
  }
  if (n < 0) return fail(c, NPFEM_ESTATE, std::string(what) + ": unsupported configuration");
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(c, NPFEM_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
  c->launches += n;
  return NPFEM_OK;
}

cudaEvent_t take_event(npfem_ctx *c) {
  if (!c->event_pool.empty()) {
    cudaEvent_t e = c->event_pool.back();
    c->event_pool.pop_back();
    return e;
  }
  cudaEvent_t e = nullptr;
  cudaEventCreate(&e);
  return e;
}

// run `launch()` (returns #kernels or <0), bracketed by events when timing is on
template <typename F>
int timed_launch(npfem_ctx *c, int kind, int type, const char *what, F launch) {
  if (!c->timing) return check_launch(c, launch(), what);
  npfem_ctx::TimedSpan sp{take_event(c), take_event(c), kind, type, 0};
  cudaEventRecord(sp.a, c->stream);
  const int n = launch();
  cudaEventRecord(sp.b, c->stream);
  sp.launches = n > 0 ? n : 0;
  c->spans.push_back(sp);
  return check_launch(c, n, what);
}

int drain_spans(npfem_ctx *c) {
  const size_t nt = c->host_types.size();
  if (c->kind_ms.size() != NPFEM_KIND_COUNT * nt) {
    c->kind_ms.assign(NPFEM_KIND_COUNT * nt, 0.0);
    c->kind_launches.assign(NPFEM_KIND_COUNT * nt, 0);
  }
  if (c->spans.empty()) return NPFEM_OK;
  NPFEM_CUDA(c, cudaStreamSynchronize(c->stream));
  for (auto &sp : c->spans) {
    float ms = 0.f;
    if (sp.launches > 0 && cudaEventElapsedTime(&ms, sp.a, sp.b) == cudaSuccess) {
      c->kind_ms[sp.kind * nt + sp.type] += ms;
      c->kind_launches[sp.kind * nt + sp.type] += sp.launches;
    }
    c->event_pool.push_back(sp.a);
    c->event_pool.push_back(sp.b);
  }
  c->spans.clear();
  cudaGetLastError();
  return NPFEM_OK;
}

void compute_layout(npfem_ctx *c) {
  auto &L = c->lay;
  const size_t es = esize(c->precision);
  size_t off = 0;
  auto take = [&](size_t bytes) {
    const size_t o = off;
    off = align_up(off + bytes);
    return o;
  };
  const size_t nt = c->host_types.size();
  for (auto &v : L.type_off) v.assign(nt, 0);
  for (int f = 0; f < F_COUNT; ++f) L.field_off[f].assign(nt, 0);
  L.origin_off.assign(nt, 0);
  L.cellid_off.assign(nt, 0);
  L.scratch_off.assign(nt, 0);
  // (1) the constant per-type tables of ALL types, (2) the create-time arena, overlaid by (3) the per-bucket state
  for (size_t t = 0; t < nt; ++t) {
    const HostTypeData &h = c->host_types[t];
    const size_t n = h.n, T = h.T, vm = h.valence_max, np = h.n_pad;
    L.type_off[0][t] = take(T * sizeof(int4));
    L.type_off[1][t] = take(T * sizeof(int4));
    L.type_off[2][t] = take(T * 4 * es);
    L.type_off[3][t] = take(T * 6 * es);
    L.type_off[4][t] = take(vm * n * sizeof(int));
    L.type_off[5][t] = take(vm * n * sizeof(int));
    L.type_off[6][t] = take((vm + 1) * n * es);
    L.type_off[7][t] = take(n * es);
    L.type_off[8][t] = take(n * es);
    L.type_off[9][t] = take(np * np * es);
    L.type_off[10][t] = take(c->precision == NPFEM_F32 ? np * np * 4 : 0);
    const bool f32 = c->precision == NPFEM_F32;
    L.type_off[11][t] = take(f32 ? T * 16 : 0);
    L.type_off[12][t] = take(f32 ? n * 16 : 0);
    L.type_off[13][t] = take(f32 ? n * 4 : 0);
    const LocalSchedule &sc = c->sched[t];
    L.type_off[14][t] = take(sc.valid ? sc.tri_words.size() * 4 : 0);
    L.type_off[15][t] = take(sc.valid ? sc.tri_consts.size() * 4 : 0);
    L.type_off[16][t] = take(sc.valid ? sc.vtx_words.size() * 4 : 0);
    L.type_off[17][t] = take(sc.valid ? sc.vtx_coef.size() * 4 : 0);
    L.type_off[18][t] = take(f32 ? np * np * 4 : 0);   // W_lo
    const QuadSchedule &qs = c->quad[t];
    L.type_off[19][t] = take(qs.valid ? qs.quad_words.size() * 4 : 0);
    L.type_off[20][t] = take(qs.valid ? qs.quad_consts.size() * 4 : 0);
    L.type_off[21][t] = take(qs.valid ? qs.vtx_words.size() * 4 : 0);
    L.type_off[22][t] = take(qs.valid ? qs.vtx_coef.size() * 4 : 0);
    const QuadMpSchedule &qm = c->quadmp[t];
    L.type_off[23][t] = take(qm.valid ? qm.quad_words.size() * 4 : 0);
    L.type_off[24][t] = take(qm.valid ? qm.quad_consts.size() * 4 : 0);
    L.type_off[25][t] = take(qm.valid ? qm.list_words.size() * 4 : 0);
    L.type_off[26][t] = take(qm.valid ? qm.vtx_slot.size() * 4 : 0);
    L.type_off[27][t] = take(qm.valid ? qm.vtx_coef.size() * 4 : 0);
    L.setup_bytes = std::max(L.setup_bytes, (2 * n * n + invert_spd_tmp_doubles(h.n)) * sizeof(double));
  }
  L.setup_off = off;
  for (size_t t = 0; t < nt; ++t) {
    const HostTypeData &h = c->host_types[t];
    const size_t np = h.n_pad;
    const bool f32 = c->precision == NPFEM_F32;
    const size_t cells = size_t(c->buckets[t].cells);
    for (int f = 0; f < F_COUNT; ++f) L.field_off[f][t] = take(f == F_XL && !f32 ? 0 : cells * 3 * np * es);
    L.origin_off[t] = take(cells * 3 * sizeof(double));
    L.cellid_off[t] = take(cells * sizeof(int64_t));
    TypeDev tmp;
    tmp.n = h.n;
    tmp.T = h.T;
    L.scratch_off[t] = take(cells ? local_generic_scratch_bytes(tmp, c->precision, c->n_sm) : 0);
  }
  L.views_off = take(nt * sizeof(BucketView));
  L.refs_all_off = take(size_t(c->n_cells) * sizeof(CellRef));
  L.refs_tmp_off = take(size_t(c->n_cells) * sizeof(CellRef));
  L.stage_a_off = take(size_t(c->total_vertices) * 3 * sizeof(double));
  L.stage_b_off = take(size_t(c->total_vertices) * 3 * sizeof(double));
  L.stage_c_off = take(size_t(c->total_vertices) * 3 * sizeof(double));
  L.total = std::max(off, align_up(L.setup_off + L.setup_bytes));
}

// ---- optional features: scratch arena ---------------------------------------------------------
constexpr int FEAT_DIAG = 0, FEAT_LS = 1, FEAT_COL = 2, FEAT_COUNT = 3;

bool ls_wants_3xtf32(const npfem_ctx *c, size_t t) {
  return c->precision == NPFEM_F32 && c->host_types[t].n_pad > 0 && c->types.size() > t && c->types[t].Hinv_tf32 &&
         global_tcgen05_supported(c->types[t]);
}

// bytes of one feature (a pure function of the context: same answer before and after the workspace is bound)
size_t feature_bytes(const npfem_ctx *c, int f) {
  const size_t es = esize(c->precision), nb = c->buckets.size();
  size_t total = 0;
  if (f == FEAT_DIAG) return align_up(size_t(NPFEM_MAX_ITERATIONS + 1) * size_t(c->n_cells ? c->n_cells : 1) * sizeof(double));
  for (size_t t = 0; t < nb; ++t) {
    const size_t cells = size_t(c->buckets[t].cells), np = size_t(c->host_types[t].n_pad);
    if (f == FEAT_LS) {
      total += align_up(4 * cells * sizeof(double)) + align_up((cells + 1) * sizeof(int)) + align_up(cells * 3 * np * es);
      if (c->precision == NPFEM_F32) total += align_up(cells * 3 * np * 4);   // g_lo of the 3xTF32 product
    } else {
      total += align_up(cells * 3 * np * sizeof(double)) + align_up(cells * np * es);
    }
  }
  if (f == FEAT_COL) total += align_up(nb * sizeof(CollisionDev));
  return total;
}

// carve a live feature out of its arena and initialise it (stream-ordered; called once per feature, never from npfem_step)
int materialise_feature(npfem_ctx *c, int f) {
  npfem_ctx::FeatureMem &m = c->feat[f];
  if (m.live) return NPFEM_OK;
  const size_t need = feature_bytes(c, f);
  if (!m.base) {
    if (c->ws && !c->ws_owned)
      return fail(c, NPFEM_ENOMEM, "the workspace is caller-owned: bind " + std::to_string(need) +
                                       " bytes of scratch for this feature first (npfem_scratch_bytes / npfem_bind_scratch)");
    void *p = nullptr;
    if (cudaMalloc(&p, need ? need : 256) != cudaSuccess) {
      cudaGetLastError();
      return fail(c, NPFEM_ENOMEM, "cannot allocate " + std::to_string(need) + " bytes of scratch");
    }
    m.base = static_cast<unsigned char *>(p);
    m.bytes = need;
    m.owned = true;
  }
  if (m.bytes < need) return fail(c, NPFEM_ENOMEM, "scratch too small for this feature: need " + std::to_string(need) + " bytes");
  // caller memory arrives with whatever it held: the padding columns of g_lo and d_old are never written by the
  // kernels but ARE read by the GEMM (a NaN there times a zero of the operator is a NaN)
  if (need) NPFEM_CUDA(c, cudaMemsetAsync(m.base, 0, need, c->stream));
  const size_t es = esize(c->precision), nb = c->buckets.size();
  unsigned char *p = m.base;
  auto take = [&](size_t bytes) { unsigned char *q = p; p += align_up(bytes); return q; };
  if (f == FEAT_DIAG) {
    c->history_dev = reinterpret_cast<double *>(take(need));
  } else if (f == FEAT_LS) {
    c->ls.assign(nb, LineSearchDev());
    for (size_t t = 0; t < nb; ++t) {
      LineSearchDev &l = c->ls[t];
      const size_t cells = size_t(c->buckets[t].cells), np = size_t(c->host_types[t].n_pad);
      l.obj0 = reinterpret_cast<double *>(take(4 * cells * sizeof(double)));
      l.obj1 = l.obj0 + cells;
      l.slope = l.obj1 + cells;
      l.alpha = l.slope + cells;
      l.done = reinterpret_cast<int *>(take((cells + 1) * sizeof(int)));   // + done[cells]: cells still searching
      l.d_old = take(cells * 3 * np * es);
      if (c->precision == NPFEM_F32) {
        float *g_lo = reinterpret_cast<float *>(take(cells * 3 * np * 4));
        // fp32 + tensor-core global step: TF32 rounding of g and H~^-1 (2^-11 per entry) spoils the search direction in
        // the stiff modes - on the violent case of tests/test_parity_gpu.py every cell ends up rejecting all step
        // lengths by iteration 11 - so the line search takes its direction from a 3xTF32 product (fp32-grade)
        if (cells && ls_wants_3xtf32(c, t)) l.g_lo = g_lo;
      }
    }
  } else {
    c->col.assign(nb, CollisionDev());
    for (size_t t = 0; t < nb; ++t) {
      const size_t slots = size_t(c->buckets[t].cells) * c->host_types[t].n_pad;
      c->col[t].targets = reinterpret_cast<double *>(take(3 * slots * sizeof(double)));
      c->col[t].stiffness = take(slots * es);
      if (slots) {
        NPFEM_CUDA(c, cudaMemsetAsync(c->col[t].targets, 0, 3 * slots * sizeof(double), c->stream));
        NPFEM_CUDA(c, cudaMemsetAsync(c->col[t].stiffness, 0, slots * es, c->stream));
      }
    }
    c->col_dev = reinterpret_cast<CollisionDev *>(take(nb * sizeof(CollisionDev)));
    NPFEM_CUDA(c, cudaMemcpyAsync(c->col_dev, c->col.data(), nb * sizeof(CollisionDev), cudaMemcpyHostToDevice, c->stream));
    NPFEM_CUDA(c, cudaStreamSynchronize(c->stream));
  }
  m.live = true;
  return NPFEM_OK;
}

// a feature was asked for: materialise it now if the workspace is ready, else when it becomes ready
int want_feature(npfem_ctx *c, int f) {
  c->feat[f].wanted = true;
  return c->ready ? materialise_feature(c, f) : NPFEM_OK;
}

template <typename T>
std::vector<T> convert(const std::vector<double> &v) {
  std::vector<T> out(v.size());
  for (size_t i = 0; i < v.size(); ++i) out[i] = T(v[i]);
  return out;
}

// upload a double vector as the compute type
int upload_real(npfem_ctx *c, size_t off, const std::vector<double> &v) {
  if (c->precision == NPFEM_F32) {
    const std::vector<float> f = convert<float>(v);
    NPFEM_CUDA(c, cudaMemcpyAsync(c->ws + off, f.data(), f.size() * 4, cudaMemcpyHostToDevice, c->stream));
    NPFEM_CUDA(c, cudaStreamSynchronize(c->stream));
  } else {
    NPFEM_CUDA(c, cudaMemcpyAsync(c->ws + off, v.data(), v.size() * 8, cudaMemcpyHostToDevice, c->stream));
    NPFEM_CUDA(c, cudaStreamSynchronize(c->stream));
  }
  return NPFEM_OK;
}

template <typename V>
int upload_raw(npfem_ctx *c, size_t off, const std::vector<V> &v) {
  if (v.empty()) return NPFEM_OK;
  NPFEM_CUDA(c, cudaMemcpyAsync(c->ws + off, v.data(), v.size() * sizeof(V), cudaMemcpyHostToDevice, c->stream));
  NPFEM_CUDA(c, cudaStreamSynchronize(c->stream));
  return NPFEM_OK;
}

// Allocate (if not bound) and fill the workspace: type tables, H~^-1, cell tables.
int ensure_ready(npfem_ctx *c) {
  if (c->ready) return NPFEM_OK;
  NPFEM_CUDA(c, cudaSetDevice(c->device));
  if (!c->ws) {
    void *p = nullptr;
    if (cudaMalloc(&p, c->lay.total ? c->lay.total : 256) != cudaSuccess) {
      cudaGetLastError();
      return fail(c, NPFEM_ENOMEM, "cannot allocate " + std::to_string(c->lay.total) + " bytes of device workspace");
    }
    c->ws = static_cast<unsigned char *>(p);
    c->ws_bytes = c->lay.total;
    c->ws_owned = true;
  }
  auto &L = c->lay;
  const size_t nt = c->host_types.size();
  c->types.assign(nt, TypeDev());
  c->views.assign(nt, BucketView());
  c->cell_id_dev.assign(nt, nullptr);
  for (size_t t = 0; t < nt; ++t) {
    const HostTypeData &h = c->host_types[t];
    TypeDev &d = c->types[t];
    d.n = h.n; d.T = h.T; d.n_pad = h.n_pad; d.valence_max = h.valence_max;
    int rc;
    if ((rc = upload_raw(c, L.type_off[0][t], h.tri))) return rc;
    if ((rc = upload_raw(c, L.type_off[1][t], h.tri_nbr))) return rc;
    if ((rc = upload_real(c, L.type_off[2][t], h.tri_rest))) return rc;
    if ((rc = upload_real(c, L.type_off[3][t], h.hinge_rest))) return rc;
    if ((rc = upload_raw(c, L.type_off[4][t], h.vtx_corner))) return rc;
    if ((rc = upload_raw(c, L.type_off[5][t], h.vtx_nbr))) return rc;
    if ((rc = upload_real(c, L.type_off[6][t], h.vtx_w))) return rc;
    if ((rc = upload_real(c, L.type_off[7][t], h.mass))) return rc;
    std::vector<double> inv_area(h.n);
    for (int v = 0; v < h.n; ++v) inv_area[v] = 1.0 / h.area_v[v];
    if ((rc = upload_real(c, L.type_off[8][t], inv_area))) return rc;
    d.tri = reinterpret_cast<const int4 *>(c->ws + L.type_off[0][t]);
    d.tri_nbr = reinterpret_cast<const int4 *>(c->ws + L.type_off[1][t]);
    d.tri_rest = c->ws + L.type_off[2][t];
    d.hinge_rest = c->ws + L.type_off[3][t];
    d.vtx_corner = reinterpret_cast<const int *>(c->ws + L.type_off[4][t]);
    d.vtx_nbr = reinterpret_cast<const int *>(c->ws + L.type_off[5][t]);
    d.vtx_w = c->ws + L.type_off[6][t];
    d.vtx_mass = c->ws + L.type_off[7][t];
    d.vtx_inv_area = c->ws + L.type_off[8][t];
    d.Hinv = c->ws + L.type_off[9][t];
    d.Hinv_tf32 = c->precision == NPFEM_F32 ? c->ws + L.type_off[10][t] : nullptr;
    const npfem_material &m = h.mat;
    d.h = h.h;
    d.B4 = m.skalak_B / 4.0;
    d.C4 = m.skalak_C / 4.0;
    d.k_b = m.k_bending;
    d.kv_over_V0 = m.k_volume / h.V0;
    d.V0 = h.V0;
    d.k_mem = m.skalak_B + 2.0 * m.skalak_C;
    d.beta_over_h = m.rayleigh_beta / h.h;
    d.inertia_coef = (1.0 + h.h * m.rayleigh_alpha) / (h.h * h.h);
    d.kappa = m.kappa_damping;
    d.gamma = d.beta_over_h / (1.0 + d.beta_over_h);
    if (c->precision == NPFEM_F32 && h.valence_max <= 8 && h.n < 65535 && 3 * h.T + 1 <= 65535) {
      // packed tables of the shared-memory local step
      std::vector<uint32_t> tri_pack(size_t(h.T) * 4), vtx_pack(size_t(h.n) * 4);
      for (int tt = 0; tt < h.T; ++tt) {
        const int32_t *v = &h.tri[4 * tt], *nb = &h.tri_nbr[4 * tt];
        tri_pack[4 * tt + 0] = uint32_t(v[0]) | (uint32_t(v[1]) << 16);
        tri_pack[4 * tt + 1] = uint32_t(v[2]) | (uint32_t(nb[0]) << 16);
        tri_pack[4 * tt + 2] = uint32_t(nb[1]) | (uint32_t(nb[2]) << 16);
        tri_pack[4 * tt + 3] = 0;
      }
      std::vector<float> coef(h.n);
      for (int v = 0; v < h.n; ++v) {
        uint32_t ids[8];
        for (int q = 0; q < 8; ++q) {
          const int32_t cid = q < h.valence_max ? h.vtx_corner[size_t(q) * h.n + v] : -1;
          ids[q] = cid >= 0 ? uint32_t(cid) : uint32_t(3 * h.T);
        }
        for (int q = 0; q < 4; ++q) vtx_pack[4 * v + q] = ids[2 * q] | (ids[2 * q + 1] << 16);
        coef[v] = float((1.0 - d.gamma) * d.inertia_coef * h.mass[v]);
      }
      if (h.T < 65536) {
        if ((rc = upload_raw(c, L.type_off[11][t], tri_pack))) return rc;
        if ((rc = upload_raw(c, L.type_off[12][t], vtx_pack))) return rc;
        if ((rc = upload_raw(c, L.type_off[13][t], coef))) return rc;
        d.tri_pack = c->ws + L.type_off[11][t];
        d.vtx_pack = c->ws + L.type_off[12][t];
        d.vtx_coef = c->ws + L.type_off[13][t];
      }
    }
    if (c->sched[t].valid) {
      const LocalSchedule &sc = c->sched[t];
      if ((rc = upload_raw(c, L.type_off[14][t], sc.tri_words))) return rc;
      if ((rc = upload_raw(c, L.type_off[15][t], sc.tri_consts))) return rc;
      if ((rc = upload_raw(c, L.type_off[16][t], sc.vtx_words))) return rc;
      if ((rc = upload_raw(c, L.type_off[17][t], sc.vtx_coef))) return rc;
      SchedDev &sd = d.sched;
      sd.valid = true;
      sd.threads = sc.threads; sd.vstride = sc.vstride; sd.tpt = sc.tpt; sd.ttri = sc.ttri; sd.maxv = sc.maxv;
      sd.n_vslots = sc.n_vslots; sd.n_tslots = sc.n_tslots; sd.n_cslots = sc.n_cslots;
      sd.vol_lane_bound = sc.vol_lane_bound;
      sd.tri_words = reinterpret_cast<const uint32_t *>(c->ws + L.type_off[14][t]);
      sd.tri_consts = reinterpret_cast<const float *>(c->ws + L.type_off[15][t]);
      sd.vtx_words = reinterpret_cast<const uint32_t *>(c->ws + L.type_off[16][t]);
      sd.vtx_coef = reinterpret_cast<const float *>(c->ws + L.type_off[17][t]);
    }
    if (c->quad[t].valid) {
      const QuadSchedule &qs = c->quad[t];
      if ((rc = upload_raw(c, L.type_off[19][t], qs.quad_words))) return rc;
      if ((rc = upload_raw(c, L.type_off[20][t], qs.quad_consts))) return rc;
      if ((rc = upload_raw(c, L.type_off[21][t], qs.vtx_words))) return rc;
      if ((rc = upload_raw(c, L.type_off[22][t], qs.vtx_coef))) return rc;
      SchedDev &qd = d.quad;
      qd.valid = true;
      qd.threads = qs.threads; qd.vstride = qs.vstride; qd.tpt = 1; qd.ttri = qs.qthreads; qd.ttri_used = qs.nq; qd.maxv = qs.maxq;
      qd.n_vslots = qs.n_vslots; qd.n_tslots = qs.n_tslots; qd.n_cslots = qs.n_cslots;
      qd.vol_lane_bound = qs.vol_lane_bound;
      qd.tri_words = reinterpret_cast<const uint32_t *>(c->ws + L.type_off[19][t]);
      qd.tri_consts = reinterpret_cast<const float *>(c->ws + L.type_off[20][t]);
      qd.vtx_words = reinterpret_cast<const uint32_t *>(c->ws + L.type_off[21][t]);
      qd.vtx_coef = reinterpret_cast<const float *>(c->ws + L.type_off[22][t]);
    }
    if (c->quadmp[t].valid) {
      const QuadMpSchedule &qm = c->quadmp[t];
      if ((rc = upload_raw(c, L.type_off[23][t], qm.quad_words))) return rc;
      if ((rc = upload_raw(c, L.type_off[24][t], qm.quad_consts))) return rc;
      if ((rc = upload_raw(c, L.type_off[25][t], qm.list_words))) return rc;
      if ((rc = upload_raw(c, L.type_off[26][t], qm.vtx_slot))) return rc;
      if ((rc = upload_raw(c, L.type_off[27][t], qm.vtx_coef))) return rc;
      QuadMpDev &md = d.quadmp;
      md.valid = true;
      md.passes = qm.passes; md.nq = qm.nq; md.maxv = qm.maxq; md.lstride = qm.lstride;
      md.n_vslots = qm.n_vslots; md.n_tslots = qm.n_tslots; md.n_cslots = qm.n_cslots;
      for (int i = 0; i < qm.passes && i < 4; ++i) md.list_len[i] = qm.list_len[i];
      md.vol_lane_bound = qm.vol_lane_bound;
      md.quad_words = reinterpret_cast<const uint32_t *>(c->ws + L.type_off[23][t]);
      md.quad_consts = reinterpret_cast<const float *>(c->ws + L.type_off[24][t]);
      md.list_words = reinterpret_cast<const uint32_t *>(c->ws + L.type_off[25][t]);
      md.vtx_slot = reinterpret_cast<const uint32_t *>(c->ws + L.type_off[26][t]);
      md.vtx_coef = reinterpret_cast<const float *>(c->ws + L.type_off[27][t]);
    }

    // dense inverse of H~ on the device (fp64), then cast/pad to the compute type.  H~, the inverse and the
    // Newton-Schulz temporaries sit in the create-time arena of the workspace (overlaid by the state fields, which
    // nothing has written yet): the library allocates no device memory of its own here
    const size_t hb = size_t(h.n) * h.n * sizeof(double);
    double *H64 = reinterpret_cast<double *>(c->ws + L.setup_off), *Hinv64 = H64 + size_t(h.n) * h.n;
    double *inv_tmp = Hinv64 + size_t(h.n) * h.n;
    cudaError_t e = cudaMemcpyAsync(H64, h.H.data(), hb, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    std::string ierr;
    double residual = 0;
    int nl = e == cudaSuccess ? launch_invert_spd(H64, Hinv64, h.n, inv_tmp, c->stream, &residual, ierr) : -1;
    if (nl >= 0) {
      nl += launch_convert_pad(Hinv64, h.n, c->ws + L.type_off[9][t], h.n_pad, c->precision, c->stream);
      if (c->precision == NPFEM_F32) {   // the tensor-core operands: W_hi = H~^-1 rounded to TF32 to nearest (internal.h,
        // tf32_rn) and W_lo = tf32(H~^-1 - W_hi) (split-operator GEMM, 3xTF32 line search)
        nl += launch_round_tf32(reinterpret_cast<const float *>(c->ws + L.type_off[9][t]),
                                reinterpret_cast<float *>(c->ws + L.type_off[10][t]), size_t(h.n_pad) * h.n_pad, c->stream);
        nl += launch_ls_split_w(reinterpret_cast<const float *>(c->ws + L.type_off[9][t]),
                                reinterpret_cast<const float *>(c->ws + L.type_off[10][t]),
                                reinterpret_cast<float *>(c->ws + L.type_off[18][t]), size_t(h.n_pad) * h.n_pad, c->stream);
        d.Hinv_lo = c->ws + L.type_off[18][t];
      }
      e = cudaStreamSynchronize(c->stream);
    }
    if (e != cudaSuccess) return fail(c, NPFEM_ECUDA, std::string("H~ inverse: ") + cudaGetErrorString(e));
    if (nl < 0) return fail(c, NPFEM_ESTATE, ierr);
    c->launches += nl;
  }
  // the create-time arena is free again: buckets, cell tables (they overlay it)
  for (size_t t = 0; t < nt; ++t) {
    const HostTypeData &h = c->host_types[t];
    int rc;
    Bucket &b = c->buckets[t];
    BucketView &bv = c->views[t];
    for (int f = 0; f < F_COUNT; ++f)
      bv.field[f] = b.field[f] = (f == F_XL && c->precision != NPFEM_F32) ? nullptr : c->ws + L.field_off[f][t];
    bv.origin = b.origin = reinterpret_cast<double *>(c->ws + L.origin_off[t]);
    bv.cells = b.cells;
    bv.n = h.n;
    bv.n_pad = h.n_pad;
    b.scratch = c->ws + L.scratch_off[t];
    c->cell_id_dev[t] = reinterpret_cast<int64_t *>(c->ws + L.cellid_off[t]);
    std::vector<int64_t> ids;
    ids.reserve(size_t(b.cells));
    for (int64_t cell = 0; cell < c->n_cells; ++cell)
      if (c->type_of_cell[cell] == int(t)) ids.push_back(cell);
    if ((rc = upload_raw(c, L.cellid_off[t], ids))) return rc;
  }
  c->views_dev = reinterpret_cast<BucketView *>(c->ws + L.views_off);
  c->refs_all_dev = reinterpret_cast<CellRef *>(c->ws + L.refs_all_off);
  c->refs_tmp_dev = reinterpret_cast<CellRef *>(c->ws + L.refs_tmp_off);
  c->stage_a = c->ws + L.stage_a_off;
  c->stage_b = c->ws + L.stage_b_off;
  c->stage_c = c->ws + L.stage_c_off;
  int rc;
  if ((rc = upload_raw(c, L.views_off, c->views))) return rc;
  std::vector<CellRef> refs(size_t(c->n_cells));
  for (int64_t cell = 0; cell < c->n_cells; ++cell)
    refs[cell] = CellRef{c->user_offset_all[cell], c->type_of_cell[cell], c->slot_of_cell[cell]};
  if ((rc = upload_raw(c, L.refs_all_off, refs))) return rc;
  c->ready = true;
  for (int f = 0; f < FEAT_COUNT; ++f)      // features asked for before the workspace existed
    if (c->feat[f].wanted && (c->feat[f].base || c->ws_owned) && (rc = materialise_feature(c, f))) return rc;
  return NPFEM_OK;
}

// Resolve a cell-id list to device CellRefs; returns element count of the packed user buffer.
int resolve_refs(npfem_ctx *c, const int64_t *cell_ids, int64_t n_ids, const CellRef **refs_dev,
                 int64_t *n_refs, int64_t *n_elems, bool mark_set) {
  if (!cell_ids) {
    *refs_dev = c->refs_all_dev;
    *n_refs = c->n_cells;
    *n_elems = c->total_vertices * 3;
    if (mark_set) {
      std::fill(c->cell_is_set.begin(), c->cell_is_set.end(), uint8_t(1));
      c->n_set = c->n_cells;
    }
    return NPFEM_OK;
  }
  if (n_ids < 0 || n_ids > c->n_cells) return fail(c, NPFEM_EINVAL, "n_ids out of range");
  std::vector<CellRef> refs(static_cast<size_t>(n_ids));
  int64_t off = 0;
  // ids must be distinct: a repeated id would make the packed buffer larger than the staging areas and let two
  // CTAs write the same cell (epoch-stamped table: O(n_ids) per call)
  if (c->seen_epoch.size() != size_t(c->n_cells)) c->seen_epoch.assign(size_t(c->n_cells), 0);
  if (++c->epoch == 0) {
    std::fill(c->seen_epoch.begin(), c->seen_epoch.end(), 0u);
    c->epoch = 1;
  }
  for (int64_t i = 0; i < n_ids; ++i) {
    const int64_t id = cell_ids[i];
    if (id < 0 || id >= c->n_cells) return fail(c, NPFEM_EINVAL, "cell id " + std::to_string(id) + " out of range");
    if (c->seen_epoch[size_t(id)] == c->epoch) return fail(c, NPFEM_EINVAL, "cell id " + std::to_string(id) + " listed twice");
    c->seen_epoch[size_t(id)] = c->epoch;
    const int t = c->type_of_cell[id];
    refs[i] = CellRef{off, t, c->slot_of_cell[id]};
    off += int64_t(3) * c->host_types[t].n;
  }
  if (mark_set)
    for (int64_t i = 0; i < n_ids; ++i)
      if (!c->cell_is_set[cell_ids[i]]) {
        c->cell_is_set[cell_ids[i]] = 1;
        ++c->n_set;
      }
  if (n_ids) {
    NPFEM_CUDA(c, cudaMemcpyAsync(c->refs_tmp_dev, refs.data(), refs.size() * sizeof(CellRef),
                                  cudaMemcpyHostToDevice, c->stream));
    NPFEM_CUDA(c, cudaStreamSynchronize(c->stream));
  }
  *refs_dev = c->refs_tmp_dev;
  *n_refs = n_ids;
  *n_elems = off;
  return NPFEM_OK;
}

// Small-batch path: does bucket t take the whole-step kernel?  ONE predicate for npfem_step and
// npfem_step_host (which must not chunk a bucket that would take it unchunked, nor let a chunk fall into it).
bool takes_fused_step(const npfem_ctx *c, size_t t) {
  const bool plain = c->precision == NPFEM_F32 && !c->diagnostics && c->ls_max_halvings == 0 && !c->col_active &&
                     c->opt_local_impl == 0 && c->opt_global_math == 0;
  return plain && c->buckets[t].cells > 0 && c->opt_fused_step != 1 && step_fused_supported(c->types[t]) &&
         (c->opt_fused_step == 2 || 2 * c->buckets[t].cells <= int64_t(3) * c->n_sm);
}

int common_checks(npfem_ctx *c, int32_t dtype, int32_t where) {
  if (!c) return NPFEM_EINVAL;
  if (c->sticky) return fail(c, NPFEM_ECUDA, "context is in a sticky CUDA error state: " + c->err);
  if (dtype != NPFEM_F32 && dtype != NPFEM_F64) return fail(c, NPFEM_EINVAL, "dtype must be NPFEM_F32 or NPFEM_F64");
  if (where != NPFEM_DEVICE && where != NPFEM_HOST) return fail(c, NPFEM_EINVAL, "where must be NPFEM_DEVICE or NPFEM_HOST");
  return NPFEM_OK;
}

}  // namespace

// =============================================================================================
extern "C" {

const char *npfem_version(void) { return "0.1.0 (sm_100a)"; }

const char *npfem_last_error(const npfem_ctx *ctx) { return ctx ? ctx->err.c_str() : g_create_error.c_str(); }

int64_t npfem_launch_count(const npfem_ctx *ctx) { return ctx ? ctx->launches : 0; }

int npfem_create(npfem_ctx **out, const npfem_cell_type *types, int32_t n_types, const int32_t *type_of_cell,
                 int64_t n_cells, double dt, int32_t precision, int32_t device, void *cuda_stream) {
  if (!out) return fail(nullptr, NPFEM_EINVAL, "out is NULL");
  *out = nullptr;
  if (!types || n_types < 1 || n_cells < 0 || (n_cells > 0 && !type_of_cell))
    return fail(nullptr, NPFEM_EINVAL, "types/type_of_cell missing or counts invalid");
  if (precision != NPFEM_F32 && precision != NPFEM_F64)
    return fail(nullptr, NPFEM_EINVAL, "precision must be NPFEM_F32 or NPFEM_F64");
  if (!(dt > 0)) return fail(nullptr, NPFEM_EINVAL, "dt must be positive");
  npfem_ctx *c = new (std::nothrow) npfem_ctx();
  if (!c) return fail(nullptr, NPFEM_ENOMEM, "out of host memory");
  c->precision = precision;
  c->device = device;
  c->stream = static_cast<cudaStream_t>(cuda_stream);
  c->dt = dt;
  c->n_cells = n_cells;
  try {
    c->host_types.resize(size_t(n_types));
    c->sched.resize(size_t(n_types));
    c->quad.resize(size_t(n_types));
    c->quadmp.resize(size_t(n_types));
    c->buckets.resize(size_t(n_types));
    for (int t = 0; t < n_types; ++t) {
      std::string err;
      const int rc = build_host_type(types[t], dt, c->host_types[t], err);
      if (rc != NPFEM_OK) {
        delete c;
        return fail(nullptr, rc, "cell type " + std::to_string(t) + ": " + err);
      }
      c->buckets[t].type = t;
      if (precision == NPFEM_F32) {
        const HostTypeData &h = c->host_types[t];
        const int tpt = h.T <= 320 ? 1 : 2;
        build_local_schedule(h, types[t].rest_positions, tpt, c->sched[t]);   // may stay invalid
        if (h.T <= 2 * 640) build_quad_schedule(h, types[t].rest_positions, c->quad[t]);   // may stay invalid
        else if (h.T <= 2 * QMP_THREADS * QMP_MAX_PASSES) build_quadmp_schedule(h, types[t].rest_positions, c->quadmp[t]);
      }
    }
    c->type_of_cell.assign(type_of_cell, type_of_cell + n_cells);
    c->slot_of_cell.resize(size_t(n_cells));
    c->user_offset_all.resize(size_t(n_cells) + 1);
    c->cell_is_set.assign(size_t(n_cells), 0);
    int64_t off = 0;
    for (int64_t cell = 0; cell < n_cells; ++cell) {
      const int t = type_of_cell[cell];
      if (t < 0 || t >= n_types) {
        delete c;
        return fail(nullptr, NPFEM_EINVAL, "type_of_cell[" + std::to_string(cell) + "] out of range");
      }
      c->slot_of_cell[cell] = int32_t(c->buckets[t].cells++);
      c->user_offset_all[cell] = off;
      off += int64_t(3) * c->host_types[t].n;
    }
    c->user_offset_all[n_cells] = off;
    c->total_vertices = off / 3;
  } catch (const std::bad_alloc &) {
    delete c;
    return fail(nullptr, NPFEM_ENOMEM, "out of host memory");
  }
  // host-side validation is done; from here on a CUDA device is required
  int n_dev = 0;
  if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev == 0) {
    cudaGetLastError();
    delete c;
    return fail(nullptr, NPFEM_ECUDA, "no CUDA device available (this library has no CPU fallback)");
  }
  if (device < 0 || device >= n_dev) {
    delete c;
    return fail(nullptr, NPFEM_EINVAL, "device ordinal out of range");
  }
  cudaDeviceProp prop;
  if (cudaSetDevice(device) != cudaSuccess || cudaGetDeviceProperties(&prop, device) != cudaSuccess) {
    delete c;
    return fail(nullptr, NPFEM_ECUDA, "cannot query the CUDA device");
  }
  if (prop.major < 10) {
    delete c;
    return fail(nullptr, NPFEM_ECUDA, "this library is built for sm_100a (B200) only");
  }
  c->n_sm = prop.multiProcessorCount;
  compute_layout(c);
  *out = c;
  return NPFEM_OK;
}

size_t npfem_workspace_bytes(const npfem_ctx *ctx) { return ctx ? ctx->lay.total : 0; }

int npfem_bind_workspace(npfem_ctx *c, void *dev_ptr, size_t bytes) {
  if (!c) return NPFEM_EINVAL;
  if (c->ready || c->ws) return fail(c, NPFEM_ESTATE, "workspace already bound or allocated");
  if (!dev_ptr || (reinterpret_cast<uintptr_t>(dev_ptr) & 255)) return fail(c, NPFEM_EINVAL, "workspace must be a 256-byte aligned device pointer");
  if (bytes < c->lay.total) return fail(c, NPFEM_ENOMEM, "workspace too small: need " + std::to_string(c->lay.total) + " bytes");
  c->ws = static_cast<unsigned char *>(dev_ptr);
  c->ws_bytes = bytes;
  c->ws_owned = false;
  return ensure_ready(c);
}

size_t npfem_scratch_bytes(const npfem_ctx *c, int32_t features) {
  if (!c) return 0;
  size_t total = 0;
  for (int f = 0; f < FEAT_COUNT; ++f)
    if (features & (1 << f)) total += feature_bytes(c, f);
  return total;
}

int npfem_bind_scratch(npfem_ctx *c, void *dev_ptr, size_t bytes, int32_t features) {
  if (!c) return NPFEM_EINVAL;
  if (features <= 0 || features >= (1 << FEAT_COUNT)) return fail(c, NPFEM_EINVAL, "features must be a non-empty mask of NPFEM_FEATURE_*");
  if (!dev_ptr || (reinterpret_cast<uintptr_t>(dev_ptr) & 255)) return fail(c, NPFEM_EINVAL, "scratch must be a 256-byte aligned device pointer");
  if (bytes < npfem_scratch_bytes(c, features))
    return fail(c, NPFEM_ENOMEM, "scratch too small: need " + std::to_string(npfem_scratch_bytes(c, features)) + " bytes");
  for (int f = 0; f < FEAT_COUNT; ++f)
    if ((features & (1 << f)) && c->feat[f].base) return fail(c, NPFEM_ESTATE, "scratch of this feature is already bound or allocated");
  unsigned char *p = static_cast<unsigned char *>(dev_ptr);
  for (int f = 0; f < FEAT_COUNT; ++f)
    if (features & (1 << f)) {
      c->feat[f].base = p;
      c->feat[f].bytes = feature_bytes(c, f);
      c->feat[f].owned = false;
      p += c->feat[f].bytes;
    }
  if (c->ready)
    for (int f = 0; f < FEAT_COUNT; ++f)
      if ((features & (1 << f)) && c->feat[f].wanted) {
        const int rc = materialise_feature(c, f);
        if (rc) return rc;
      }
  return NPFEM_OK;
}

int npfem_set_option(npfem_ctx *c, int32_t option, int64_t value) {
  if (!c) return NPFEM_EINVAL;
  switch (option) {
    case NPFEM_OPT_DIAGNOSTICS: {
      if (value != 0) {   // the objective history needs scratch: bound by the caller or allocated here, not in npfem_step
        const int rc = want_feature(c, FEAT_DIAG);
        if (rc) return rc;
      }
      c->diagnostics = value != 0;
      return NPFEM_OK;
    }
    case NPFEM_OPT_GLOBAL_STEP_MATH:
      if (value < 0 || value > 2) return fail(c, NPFEM_EINVAL, "global-step math must be 0 (TF32), 1 (FP32) or 2 (TF32, split operator)");
      c->opt_global_math = value;
      return NPFEM_OK;
    case NPFEM_OPT_LOCAL_STEP_IMPL:
      if (value < 0 || value > 6) return fail(c, NPFEM_EINVAL, "local-step impl must be 0 ... 6");
      c->opt_local_impl = value;
      return NPFEM_OK;
    case NPFEM_OPT_KERNEL_TIMING: c->timing = value != 0; return NPFEM_OK;
    case NPFEM_OPT_FORCE_MEDIAN_FILTER: c->median_filter = value != 0; return NPFEM_OK;
    case NPFEM_OPT_FUSED_STEP:
      if (value < 0 || value > 2) return fail(c, NPFEM_EINVAL, "fused-step option must be 0, 1 or 2");
      c->opt_fused_step = value;
      return NPFEM_OK;
    case NPFEM_OPT_UPDATE_MODE:   // kept for old callers: the product-out mode (2) was measured slower and is gone
      if (value < 0 || value > 1) return fail(c, NPFEM_EINVAL, "update mode must be 0 or 1 (the GEMM epilogue updates d in place)");
      return NPFEM_OK;
    default: return fail(c, NPFEM_EINVAL, "unknown option");
  }
}

int npfem_set_state(npfem_ctx *c, const int64_t *cell_ids, int64_t n_ids, const void *positions,
                    const void *velocities, int32_t dtype, int32_t where) {
  int rc = common_checks(c, dtype, where);
  if (rc) return rc;
  if (!positions) return fail(c, NPFEM_EINVAL, "positions is NULL");
  if ((rc = ensure_ready(c))) return rc;
  PackArgs a{};
  int64_t n_elems = 0;
  if ((rc = resolve_refs(c, cell_ids, n_ids, &a.refs, &a.n_refs, &n_elems, true))) return rc;
  a.io_dtype = dtype;
  a.src_a = positions;
  a.src_b = velocities;
  if (where == NPFEM_HOST && n_elems) {
    const size_t bytes = size_t(n_elems) * (dtype == NPFEM_F32 ? 4 : 8);
    NPFEM_CUDA(c, cudaMemcpyAsync(c->stage_a, positions, bytes, cudaMemcpyHostToDevice, c->stream));
    a.src_a = c->stage_a;
    if (velocities) {
      NPFEM_CUDA(c, cudaMemcpyAsync(c->stage_b, velocities, bytes, cudaMemcpyHostToDevice, c->stream));
      a.src_b = c->stage_b;
    }
  }
  if ((rc = check_launch(c, launch_set_state(c->views_dev, a, c->precision, c->stream), "set_state"))) return rc;
  if (where == NPFEM_HOST) NPFEM_CUDA(c, cudaStreamSynchronize(c->stream));
  return NPFEM_OK;
}

int npfem_set_forces(npfem_ctx *c, const int64_t *cell_ids, int64_t n_ids, const void *forces, int32_t dtype,
                     int32_t where) {
  int rc = common_checks(c, dtype, where);
  if (rc) return rc;
  if (!forces) return fail(c, NPFEM_EINVAL, "forces is NULL");
  if ((rc = ensure_ready(c))) return rc;
  PackArgs a{};
  int64_t n_elems = 0;
  if ((rc = resolve_refs(c, cell_ids, n_ids, &a.refs, &a.n_refs, &n_elems, false))) return rc;
  a.io_dtype = dtype;
  a.src_a = forces;
  if (where == NPFEM_HOST && n_elems) {
    const size_t bytes = size_t(n_elems) * (dtype == NPFEM_F32 ? 4 : 8);
    NPFEM_CUDA(c, cudaMemcpyAsync(c->stage_a, forces, bytes, cudaMemcpyHostToDevice, c->stream));
    a.src_a = c->stage_a;
  }
  if ((rc = check_launch(c, launch_set_forces(c->views_dev, a, c->precision, c->stream), "set_forces"))) return rc;
  if (c->median_filter)
    for (size_t t = 0; t < c->buckets.size(); ++t)
      if (c->buckets[t].cells &&
          (rc = check_launch(c, launch_median_filter(c->views_dev, a.refs, a.n_refs, int(t), c->types[t], c->precision, c->stream),
                             "median filter")))
        return rc;
  if (where == NPFEM_HOST) NPFEM_CUDA(c, cudaStreamSynchronize(c->stream));
  return NPFEM_OK;
}

int npfem_get_state(npfem_ctx *c, const int64_t *cell_ids, int64_t n_ids, void *positions, void *velocities,
                    int32_t dtype, int32_t where) {
  int rc = common_checks(c, dtype, where);
  if (rc) return rc;
  if (!c->ready || c->n_set != c->n_cells) return fail(c, NPFEM_ESTATE, "get_state before every cell has been given a state");
  PackArgs a{};
  int64_t n_elems = 0;
  if ((rc = resolve_refs(c, cell_ids, n_ids, &a.refs, &a.n_refs, &n_elems, false))) return rc;
  a.io_dtype = dtype;
  a.dst_a = positions;
  a.dst_b = velocities;
  if (where == NPFEM_HOST) {
    a.dst_a = positions ? c->stage_a : nullptr;
    a.dst_b = velocities ? c->stage_b : nullptr;
  }
  if ((rc = check_launch(c, launch_get_state(c->views_dev, a, c->precision, c->stream), "get_state"))) return rc;
  if (where == NPFEM_HOST) {
    const size_t bytes = size_t(n_elems) * (dtype == NPFEM_F32 ? 4 : 8);
    if (positions && bytes) NPFEM_CUDA(c, cudaMemcpyAsync(positions, c->stage_a, bytes, cudaMemcpyDeviceToHost, c->stream));
    if (velocities && bytes) NPFEM_CUDA(c, cudaMemcpyAsync(velocities, c->stage_b, bytes, cudaMemcpyDeviceToHost, c->stream));
    NPFEM_CUDA(c, cudaStreamSynchronize(c->stream));
  }
  return NPFEM_OK;
}

int npfem_step(npfem_ctx *c, int32_t n_iterations) {
  if (!c) return NPFEM_EINVAL;
  if (c->sticky) return fail(c, NPFEM_ECUDA, "context is in a sticky CUDA error state: " + c->err);
  if (n_iterations < 1 || n_iterations > NPFEM_MAX_ITERATIONS) return fail(c, NPFEM_EINVAL, "n_iterations out of range");
  if (!c->ready || c->n_set != c->n_cells) return fail(c, NPFEM_ESTATE, "step before every cell has been given a state");
  int rc;
  const size_t nb = c->buckets.size();
  // the objective history lives in the scratch arena (feature DIAGNOSTICS, NPFEM_MAX_ITERATIONS + 1 rows):
  // nothing is allocated here
  c->history_entries = c->diagnostics ? n_iterations + 1 : 0;
  if (c->diagnostics && !c->feat[FEAT_DIAG].live) return fail(c, NPFEM_ESTATE, "diagnostics are on but their scratch is not bound");
  auto diag = [&](int row) -> int {
    for (size_t t = 0; t < nb; ++t) {
      double *out = c->history_dev + size_t(row) * c->n_cells;
      int r = check_launch(c, launch_objective(c->types[t], c->views[t], c->cell_id_dev[t], out, nullptr, c->precision, c->n_sm, c->stream),
                           "objective");
      if (r) return r;
      if (c->col_active &&
          (r = check_launch(c, launch_collision_energy(c->views[t], c->col[t], c->cell_id_dev[t], out, nullptr, c->precision,
                                                       c->stream), "collision energy")))
        return r;
    }
    return NPFEM_OK;
  };
  if (c->spans.size() > 200000 && (rc = drain_spans(c))) return rc;
  // Small-batch path: a bucket with only a few cells per SM runs its whole step in one
  // kernel, one CTA per cell (step_fused.cu); everything else goes through the batched kernels below.
  std::vector<char> whole(nb, 0);
  for (size_t t = 0; t < nb; ++t) {
    whole[t] = takes_fused_step(c, t);
    if (whole[t] && (rc = timed_launch(c, NPFEM_KIND_FUSED_STEP, int(t), "fused step", [&] {
                       return launch_step_fused(c->types[t], c->views[t], c->n_sm, n_iterations, c->v_max, c->stream); })))
      return rc;
  }
  for (size_t t = 0; t < nb; ++t)
    if (!whole[t] && (rc = timed_launch(c, NPFEM_KIND_PROLOGUE, int(t), "prologue", [&] {
           return launch_prologue(c->types[t], c->views[t], c->precision, c->stream); })))
      return rc;
  const bool ls_on = c->ls_max_halvings > 0;
  if (ls_on && !c->feat[FEAT_LS].live) return fail(c, NPFEM_ESTATE, "the line search is on but its scratch is not bound");
  // which GEMM a bucket takes is decided HERE, before anything is launched: the tcgen05 kernel when the context is
  // fp32, the option asks for TF32 and the shape is supported; otherwise the SIMT kernel, reported as its own kind
  // (NPFEM_KIND_GLOBAL_SIMT).  A tensor-core launch that fails is an error, never a silent fallback.
  std::vector<char> use_tc(nb, 0);
  for (size_t t = 0; t < nb; ++t)
    use_tc[t] = c->precision == NPFEM_F32 && c->opt_global_math != 1 && global_tcgen05_supported(c->types[t]);
  // g feeds the TF32 tensor-core GEMM: the local step stores it already rounded to nearest (the line search
  // then takes its slope and gradient norm from the rounded gradient: 2^-12 relative per entry, random sign)
  for (size_t t = 0; t < nb; ++t)
    c->views[t].g_tf32 = !ls_on && use_tc[t];
  for (int k = 0; k < n_iterations; ++k) {
    if (c->diagnostics && (rc = diag(k))) return rc;
    for (size_t t = 0; t < nb; ++t) {
      if (whole[t]) continue;
      // the line search needs the FULL gradient: fp32 contexts take the fast kernels' reduced gradient and add the
      // damping part to it (launch_damping_grad), fp64 contexts take the generic kernel
      const bool f32 = c->precision == NPFEM_F32 &&
                       (!ls_on || size_t(24) * size_t(c->types[t].n) <= size_t(200) * 1024);
      const bool quad = f32 && (c->opt_local_impl == 0 || c->opt_local_impl == 5) && local_quad_supported(c->types[t]);
      const bool quadmp = f32 && !quad && (c->opt_local_impl == 0 || c->opt_local_impl == 6) && local_quadmp_supported(c->types[t]);
      const bool sched = f32 && !quad && !quadmp && (c->opt_local_impl == 0 || c->opt_local_impl == 3) && local_sched_supported(c->types[t]);
      const bool fast = f32 && !quad && !quadmp && !sched && (c->opt_local_impl == 0 || c->opt_local_impl == 2) && local_smem_supported(c->types[t]);
      const bool big = f32 && !quad && !quadmp && !sched && !fast && (c->opt_local_impl == 0 || c->opt_local_impl == 4) && local_big_supported(c->types[t]);
      const bool reduced = quad || quadmp || sched || fast || big;
      const double d_scale = reduced && !ls_on ? 1.0 - c->types[t].gamma : 1.0;
      const BucketView &lv = c->views[t];
      if ((rc = timed_launch(c, NPFEM_KIND_LOCAL, int(t), "local step", [&] {
             if (quad) return launch_local_quad(c->types[t], lv, c->n_sm, c->stream);
             if (quadmp) return launch_local_quadmp(c->types[t], lv, c->n_sm, c->stream);
             if (sched) return launch_local_sched(c->types[t], lv, c->n_sm, c->stream);
             if (fast) return launch_local_smem(c->types[t], lv, c->n_sm, c->stream);
             if (big) return launch_local_big(c->types[t], lv, c->n_sm, c->stream);
             return launch_local_generic(c->types[t], lv, c->buckets[t].scratch, c->precision, c->n_sm,
                                         c->stream); })))
        return rc;
      // 3xTF32 operands of the line search's global step: split by the damping kernel, unless the collision term is
      // still to come or the generic kernel ran (then by launch_ls_split_g just before the GEMMs)
      const bool split_early = ls_on && reduced && !c->col_active && use_tc[t] && c->ls[t].g_lo;
      if (ls_on && reduced && (rc = timed_launch(c, NPFEM_KIND_LOCAL, int(t), "damping gradient", [&] {
                                 return launch_damping_grad(c->types[t], c->views[t], split_early ? c->ls[t].g_lo : nullptr,
                                                            c->n_sm, c->stream); })))
        return rc;
      if (c->col_active && c->buckets[t].cells &&
          (rc = timed_launch(c, NPFEM_KIND_LOCAL, int(t), "collision gradient", [&] {
             return launch_collision_grad(c->views[t], c->col[t], c->precision, c->stream); })))
        return rc;
      if (ls_on && c->buckets[t].cells) {
        // g(d) of every cell and a copy of d before the global step overwrites it
        const size_t bytes = size_t(c->buckets[t].cells) * 3 * c->types[t].n_pad * esize(c->precision);
        // (first iteration only: ls_accept leaves the objective of the accepted trial point in obj0)
        if (k == 0 && (rc = timed_launch(c, NPFEM_KIND_LINE_SEARCH, int(t), "line search: objective", [&] {
               int nl = launch_objective(c->types[t], c->views[t], nullptr, c->ls[t].obj0, nullptr, c->precision, c->n_sm, c->stream);
               if (c->col_active)
                 nl += launch_collision_energy(c->views[t], c->col[t], nullptr, c->ls[t].obj0, nullptr, c->precision, c->stream);
               return nl; })))
          return rc;
        NPFEM_CUDA(c, cudaMemcpyAsync(c->ls[t].d_old, c->views[t].field[F_D], bytes, cudaMemcpyDeviceToDevice, c->stream));
      }
      const bool tc3 = ls_on && use_tc[t] && c->ls[t].g_lo;
      if ((rc = timed_launch(c, use_tc[t] ? NPFEM_KIND_GLOBAL : NPFEM_KIND_GLOBAL_SIMT, int(t), "global step", [&] {
             if (tc3) {                         // 3xTF32: d <- d - (g_hi W_hi + g_lo W_hi + g_hi W_lo), one K-concatenated GEMM
               const LineSearchDev &l = c->ls[t];
               const size_t count = size_t(c->buckets[t].cells) * 3 * c->types[t].n_pad;
               int nl = split_early ? 0 : launch_ls_split_g(static_cast<float *>(c->views[t].field[F_G]), l.g_lo, count, c->stream);
               const int n1 = launch_global_tcgen05(c->types[t], c->views[t], c->n_sm, 1.0, c->stream, l.g_lo, c->types[t].Hinv_lo);
               return n1 < 0 ? n1 : nl + n1;
             }
             if (use_tc[t])   // option 2: [g g] . [W_hi; W_lo], the operator to fp32 accuracy at twice the tensor work
               return launch_global_tcgen05(c->types[t], c->views[t], c->n_sm, d_scale, c->stream, nullptr,
                                            c->opt_global_math == 2 ? c->types[t].Hinv_lo : nullptr);
             return launch_global_simt(c->types[t], c->views[t], c->precision, d_scale, c->stream); })))
        return rc;
      if (ls_on && c->buckets[t].cells) {
        if ((rc = timed_launch(c, NPFEM_KIND_LINE_SEARCH, int(t), "line search", [&] {
               int nl = launch_ls_init(c->views[t], c->ls[t], c->ls_tol, c->precision, c->stream);
               if (nl < 0) return nl;
               for (int l = 0; l <= c->ls_max_halvings; ++l) {
                 nl += launch_objective(c->types[t], c->views[t], nullptr, c->ls[t].obj1, c->ls[t].done, c->precision, c->n_sm, c->stream);
                 if (c->col_active)
                   nl += launch_collision_energy(c->views[t], c->col[t], nullptr, c->ls[t].obj1, c->ls[t].done, c->precision,
                                                 c->stream);
                 nl += launch_ls_accept(c->views[t], c->ls[t], c->ls_c1, l == c->ls_max_halvings, c->precision, c->stream);
               }
               return nl; })))
          return rc;
        c->ls_ran = true;
      }
    }
  }
  if (c->diagnostics && (rc = diag(n_iterations))) return rc;
  for (size_t t = 0; t < nb; ++t)
    if (!whole[t] && (rc = timed_launch(c, NPFEM_KIND_EPILOGUE, int(t), "epilogue", [&] {
           return launch_epilogue(c->types[t], c->views[t], c->precision, c->v_max, c->stream); })))
      return rc;
  return NPFEM_OK;
}

// One time step with HOST buffers, pipelined (include/npfem.h).  Cells are independent within a step
// and a range of cell ids is one contiguous slab of every bucket and of the user
// buffers, so the population is cut into chunks and chunk i's solver kernels run while chunk i+1's
// forces come in and chunk i-1's state goes out, on two copy streams (PCIe is full duplex).
int npfem_step_host(npfem_ctx *c, const void *forces, int32_t n_iterations, void *positions, void *velocities,
                    int32_t dtype, int32_t n_chunks) {
  int rc = common_checks(c, dtype, NPFEM_HOST);
  if (rc) return rc;
  if (!forces || !positions || !velocities) return fail(c, NPFEM_EINVAL, "forces / positions / velocities is NULL");
  if (n_chunks < 0 || n_chunks > 64) return fail(c, NPFEM_EINVAL, "n_chunks must be in 0..64 (0 = auto)");
  if (n_iterations < 1 || n_iterations > NPFEM_MAX_ITERATIONS) return fail(c, NPFEM_EINVAL, "n_iterations out of range");
  if (!c->ready || c->n_set != c->n_cells) return fail(c, NPFEM_ESTATE, "step before every cell has been given a state");
  const size_t es = dtype == NPFEM_F32 ? 4 : 8;
  const int64_t total = c->total_vertices * 3;
  if (n_chunks == 0) n_chunks = int32_t(std::min<int64_t>(16, std::max<int64_t>(1, int64_t(total * es) / (48 << 20))));   // auto: <= 16
  n_chunks = int32_t(std::max<int64_t>(1, std::min<int64_t>(n_chunks, c->n_cells)));
  // per-cell reductions over the whole bucket (history rows, line-search state, collision tables) are
  // indexed by bucket slot: those modes take the unchunked sequence
  // the small-batch whole-step kernel is chosen by bucket size: a bucket that would take it unchunked is small
  // enough not to be worth chunking, and no chunk may fall into it when the whole bucket would not
  bool small_batch = false;      // the SAME predicate npfem_step uses (fp64 contexts, option-forced kernels ... never take it)
  for (size_t t = 0; t < c->buckets.size(); ++t) small_batch = small_batch || takes_fused_step(c, t);
  if (c->diagnostics || c->ls_max_halvings > 0 || c->col_active || c->median_filter || small_batch || n_chunks == 1) {
    if ((rc = npfem_set_forces(c, nullptr, 0, forces, dtype, NPFEM_HOST))) return rc;
    if ((rc = npfem_step(c, n_iterations))) return rc;
    return npfem_get_state(c, nullptr, 0, positions, velocities, dtype, NPFEM_HOST);
  }
  if (!c->h2d_stream) {
    NPFEM_CUDA(c, cudaStreamCreateWithFlags(&c->h2d_stream, cudaStreamNonBlocking));
    NPFEM_CUDA(c, cudaStreamCreateWithFlags(&c->d2h_stream, cudaStreamNonBlocking));
  }
  while (c->io_events.size() < size_t(2 * n_chunks + 1)) {
    cudaEvent_t e;
    NPFEM_CUDA(c, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    c->io_events.push_back(e);
  }
  const size_t nb = c->buckets.size();
  const std::vector<BucketView> full_views = c->views;
  std::vector<int64_t> full_cells(nb), slot0(nb, 0);
  for (size_t t = 0; t < nb; ++t) full_cells[t] = c->buckets[t].cells;
  auto restore = [&] {
    c->views = full_views;
    for (size_t t = 0; t < nb; ++t) c->buckets[t].cells = full_cells[t];
  };
  // the pipeline proper; on any failure the copy streams are drained before the call returns (the caller's host
  // buffers must not have copies in flight once it has the error code in hand) and the views are restored
  auto pipeline = [&]() -> int {
    // the copy-in stream starts after whatever the caller's stream still has in flight on the staging buffers
    cudaEvent_t ev_start = c->io_events[size_t(2 * n_chunks)];
    NPFEM_CUDA(c, cudaEventRecord(ev_start, c->stream));
    NPFEM_CUDA(c, cudaStreamWaitEvent(c->h2d_stream, ev_start, 0));
    NPFEM_CUDA(c, cudaStreamWaitEvent(c->d2h_stream, ev_start, 0));
    const unsigned char *f_host = static_cast<const unsigned char *>(forces);
    unsigned char *x_host = static_cast<unsigned char *>(positions), *v_host = static_cast<unsigned char *>(velocities);
    unsigned char *sa = static_cast<unsigned char *>(c->stage_a), *sb = static_cast<unsigned char *>(c->stage_b),
                  *sc = static_cast<unsigned char *>(c->stage_c);
    // all copies in are queued first: the copy engine runs ahead of the solver as far as it can
    for (int i = 0; i < n_chunks; ++i) {
      const int64_t c0 = c->n_cells * i / n_chunks, c1 = c->n_cells * (i + 1) / n_chunks;
      const size_t b0 = size_t(c->user_offset_all[c0]) * es, b1 = size_t(c->user_offset_all[c1]) * es;
      NPFEM_CUDA(c, cudaMemcpyAsync(sc + b0, f_host + b0, b1 - b0, cudaMemcpyHostToDevice, c->h2d_stream));
      NPFEM_CUDA(c, cudaEventRecord(c->io_events[size_t(i)], c->h2d_stream));
    }
    for (int i = 0; i < n_chunks; ++i) {
      const int64_t c0 = c->n_cells * i / n_chunks, c1 = c->n_cells * (i + 1) / n_chunks;
      const size_t b0 = size_t(c->user_offset_all[c0]) * es, b1 = size_t(c->user_offset_all[c1]) * es;
      std::vector<int64_t> count(nb, 0);
      for (int64_t cell = c0; cell < c1; ++cell) ++count[size_t(c->type_of_cell[cell])];
      PackArgs a{};
      a.refs = c->refs_all_dev + c0;
      a.n_refs = c1 - c0;
      a.io_dtype = dtype;
      a.src_a = sc;
      NPFEM_CUDA(c, cudaStreamWaitEvent(c->stream, c->io_events[size_t(i)], 0));
      if ((rc = check_launch(c, launch_set_forces(c->views_dev, a, c->precision, c->stream), "set_forces"))) return rc;
      for (size_t t = 0; t < nb; ++t) {
        BucketView bv = full_views[t];
        const size_t shift = size_t(slot0[t]) * 3 * size_t(bv.n_pad) * esize(c->precision);
        for (int f = 0; f < F_COUNT; ++f)
          if (bv.field[f]) bv.field[f] = static_cast<unsigned char *>(bv.field[f]) + shift;   // F_XL is null in fp64 contexts
        bv.origin += slot0[t] * 3;
        bv.cells = count[t];
        c->views[t] = bv;
        c->buckets[t].cells = count[t];
      }
      const int64_t keep_fused = c->opt_fused_step;
      c->opt_fused_step = 1;                       // see small_batch above: chunks take the kernels the whole bucket takes
      rc = npfem_step(c, n_iterations);
      c->opt_fused_step = keep_fused;
      restore();
      if (rc) return rc;
      for (size_t t = 0; t < nb; ++t) slot0[t] += count[t];
      PackArgs g{};
      g.refs = c->refs_all_dev + c0;
      g.n_refs = c1 - c0;
      g.io_dtype = dtype;
      g.dst_a = sa;
      g.dst_b = sb;
      if ((rc = check_launch(c, launch_get_state(c->views_dev, g, c->precision, c->stream), "get_state"))) return rc;
      cudaEvent_t packed = c->io_events[size_t(n_chunks + i)];
      NPFEM_CUDA(c, cudaEventRecord(packed, c->stream));
      NPFEM_CUDA(c, cudaStreamWaitEvent(c->d2h_stream, packed, 0));
      NPFEM_CUDA(c, cudaMemcpyAsync(x_host + b0, sa + b0, b1 - b0, cudaMemcpyDeviceToHost, c->d2h_stream));
      NPFEM_CUDA(c, cudaMemcpyAsync(v_host + b0, sb + b0, b1 - b0, cudaMemcpyDeviceToHost, c->d2h_stream));
    }
    NPFEM_CUDA(c, cudaStreamSynchronize(c->d2h_stream));
    NPFEM_CUDA(c, cudaStreamSynchronize(c->stream));
    return NPFEM_OK;
  };
  rc = pipeline();
  if (rc) {
    restore();
    cudaStreamSynchronize(c->h2d_stream);
    cudaStreamSynchronize(c->d2h_stream);
    cudaStreamSynchronize(c->stream);
    cudaGetLastError();
  }
  return rc;
}

int npfem_set_line_search(npfem_ctx *c, int32_t max_halvings, double armijo_c1, double grad_tol) {
  if (!c) return NPFEM_EINVAL;
  if (max_halvings < 0 || max_halvings > 30 || !(armijo_c1 >= 0) || !(armijo_c1 < 1) || !(grad_tol >= 0))
    return fail(c, NPFEM_EINVAL, "line search: 0 <= max_halvings <= 30, 0 <= armijo_c1 < 1, grad_tol >= 0");
  if (max_halvings > 0) {   // per-cell search state, d_old, 3xTF32 operands: scratch, bound by the caller or allocated here
    const int rc = want_feature(c, FEAT_LS);
    if (rc) return rc;
  }
  c->ls_max_halvings = max_halvings;
  c->ls_c1 = armijo_c1;
  c->ls_tol = grad_tol;
  return NPFEM_OK;
}

int npfem_set_collisions(npfem_ctx *c, const int64_t *cell_ids, int64_t n_ids, const void *targets, const void *stiffness,
                         int32_t dtype, int32_t where) {
  int rc = common_checks(c, dtype, where);
  if (rc) return rc;
  if (!targets || !stiffness) return fail(c, NPFEM_EINVAL, "targets / stiffness is NULL");
  if (!c->ready || c->n_set != c->n_cells) return fail(c, NPFEM_ESTATE, "set_collisions before every cell has been given a state");
  if ((rc = want_feature(c, FEAT_COL))) return rc;   // tables in the scratch arena (zeroed when first carved)
  PackArgs a{};
  int64_t n_elems = 0;
  if ((rc = resolve_refs(c, cell_ids, n_ids, &a.refs, &a.n_refs, &n_elems, false))) return rc;
  a.io_dtype = dtype;
  a.src_a = targets;
  a.src_b = stiffness;
  if (where == NPFEM_HOST && n_elems) {
    const size_t bytes = size_t(n_elems) * (dtype == NPFEM_F32 ? 4 : 8);
    NPFEM_CUDA(c, cudaMemcpyAsync(c->stage_a, targets, bytes, cudaMemcpyHostToDevice, c->stream));
    NPFEM_CUDA(c, cudaMemcpyAsync(c->stage_b, stiffness, bytes / 3, cudaMemcpyHostToDevice, c->stream));
    a.src_a = c->stage_a;
    a.src_b = c->stage_b;
  }
  if ((rc = check_launch(c, launch_set_collisions(c->views_dev, c->col_dev, a, c->precision, c->stream), "set_collisions")))
    return rc;
  if (where == NPFEM_HOST) NPFEM_CUDA(c, cudaStreamSynchronize(c->stream));
  c->col_active = true;
  return NPFEM_OK;
}

int npfem_clear_collisions(npfem_ctx *c) {
  if (!c) return NPFEM_EINVAL;
  if (c->sticky) return fail(c, NPFEM_ECUDA, "context is in a sticky CUDA error state: " + c->err);
  for (size_t t = 0; t < c->col.size() && c->feat[FEAT_COL].live; ++t) {
    const size_t slots = size_t(c->buckets[t].cells) * c->types[t].n_pad;
    if (slots) NPFEM_CUDA(c, cudaMemsetAsync(c->col[t].stiffness, 0, slots * esize(c->precision), c->stream));
  }
  c->col_active = false;
  return NPFEM_OK;
}

int npfem_set_velocity_cap(npfem_ctx *c, double v_max) {
  if (!c) return NPFEM_EINVAL;
  if (!(v_max >= 0)) return fail(c, NPFEM_EINVAL, "velocity cap must be >= 0 (0 = off)");
  c->v_max = v_max;
  return NPFEM_OK;
}

int npfem_get_step_lengths(npfem_ctx *c, double *alpha) {
  if (!c || !alpha) return NPFEM_EINVAL;
  if (c->sticky) return fail(c, NPFEM_ECUDA, "context is in a sticky CUDA error state: " + c->err);
  if (!c->ls_ran) return fail(c, NPFEM_ESTATE, "no step lengths: enable npfem_set_line_search before npfem_step");
  std::vector<std::vector<double>> per_bucket(c->buckets.size());
  for (size_t t = 0; t < c->buckets.size(); ++t) {
    per_bucket[t].resize(size_t(c->buckets[t].cells));
    if (c->buckets[t].cells)
      NPFEM_CUDA(c, cudaMemcpyAsync(per_bucket[t].data(), c->ls[t].alpha, per_bucket[t].size() * sizeof(double),
                                    cudaMemcpyDeviceToHost, c->stream));
  }
  NPFEM_CUDA(c, cudaStreamSynchronize(c->stream));
  for (int64_t cell = 0; cell < c->n_cells; ++cell) alpha[cell] = per_bucket[c->type_of_cell[cell]][c->slot_of_cell[cell]];
  return NPFEM_OK;
}

int npfem_get_kernel_times(npfem_ctx *c, double *ms, int64_t *launches, int32_t reset) {
  if (!c) return NPFEM_EINVAL;
  if (c->sticky) return fail(c, NPFEM_ECUDA, "context is in a sticky CUDA error state: " + c->err);
  const int rc = drain_spans(c);
  if (rc) return rc;
  const size_t cnt = c->kind_ms.size();
  if (ms) std::copy(c->kind_ms.begin(), c->kind_ms.end(), ms);
  if (launches) std::copy(c->kind_launches.begin(), c->kind_launches.end(), launches);
  if (reset) {
    std::fill(c->kind_ms.begin(), c->kind_ms.end(), 0.0);
    std::fill(c->kind_launches.begin(), c->kind_launches.end(), 0);
  }
  (void)cnt;
  return NPFEM_OK;
}

int npfem_get_objective(npfem_ctx *c, double *history, int32_t max_entries, int32_t *n_entries, int32_t *monotone,
                        int32_t where) {
  int rc = common_checks(c, NPFEM_F64, where);
  if (rc) return rc;
  if (!c->history_entries) return fail(c, NPFEM_ESTATE, "no objective history: enable NPFEM_OPT_DIAGNOSTICS before npfem_step");
  const int rows = std::min<int>(max_entries, c->history_entries);
  if (n_entries) *n_entries = c->history_entries;
  const cudaMemcpyKind kind = where == NPFEM_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice;
  if (history && rows > 0 && c->n_cells)
    NPFEM_CUDA(c, cudaMemcpyAsync(history, c->history_dev, size_t(rows) * c->n_cells * sizeof(double), kind, c->stream));
  if (monotone && c->n_cells) {
    int32_t *flags = where == NPFEM_HOST ? static_cast<int32_t *>(c->stage_a) : monotone;
    if ((rc = check_launch(c, launch_monotone_flags(c->history_dev, c->history_entries, c->n_cells, flags, c->stream), "monotone")))
      return rc;
    if (where == NPFEM_HOST)
      NPFEM_CUDA(c, cudaMemcpyAsync(monotone, flags, size_t(c->n_cells) * sizeof(int32_t), cudaMemcpyDeviceToHost, c->stream));
  }
  if (where == NPFEM_HOST) NPFEM_CUDA(c, cudaStreamSynchronize(c->stream));
  return NPFEM_OK;
}

int npfem_local_schedule_stats(const npfem_cell_type *type, double dt, double *stats, int32_t n_stats) {
  if (!type || !stats || n_stats < 10 || !(dt > 0)) return fail(nullptr, NPFEM_EINVAL, "type/stats missing, n_stats < 10 or dt <= 0");
  std::fill(stats, stats + n_stats, 0.0);
  HostTypeData h;
  std::string err;
  const int rc = build_host_type(*type, dt, h, err);
  if (rc != NPFEM_OK) return fail(nullptr, rc, err);
  LocalSchedule sc;
  const auto t0 = std::chrono::steady_clock::now();
  if (!build_local_schedule(h, type->rest_positions, h.T <= 320 ? 1 : 2, sc)) return NPFEM_OK;
  stats[9] = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
  stats[0] = 1;
  stats[1] = sc.threads;
  stats[2] = sc.tpt;
  stats[3] = sc.wf_vertex;
  stats[4] = sc.wf_normal;
  stats[8] = double(sc.n_vslots + sc.n_tslots + sc.n_cslots) * 16.0;
  // ---- decode the tables and check them against the mesh ------------------------------------
  auto lo = [](uint32_t w) { return int(w & 0xffffu) / 16; };
  auto hi = [](uint32_t w) { return int(w >> 16) / 16; };
  bool ok = true;
  std::vector<int> vslot(size_t(h.n)), tslot(size_t(h.T)), seen_v(size_t(sc.n_vslots), 0), seen_t(size_t(sc.n_tslots), 0),
      seen_c(size_t(sc.n_cslots), 0);
  for (int v = 0; v < h.n; ++v) {
    vslot[v] = lo(sc.vtx_words[v]);
    ok &= vslot[v] < sc.n_vslots && !seen_v[vslot[v]]++;
  }
  auto W = [&](int t, int q) { return sc.tri_words[(size_t(t / sc.ttri) * 5 + q) * sc.threads + t % sc.ttri]; };
  for (int t = 0; t < h.T; ++t) {
    tslot[t] = hi(W(t, 4));
    ok &= tslot[t] < sc.n_tslots && !seen_t[tslot[t]]++;
  }
  std::vector<std::vector<int>> corner_slots(size_t(h.n));     // per vertex: slots its triangles write
  double worst_store = 0, worst_gather = 0;
  for (int t = 0; t < h.T; ++t) {
    const int vs[3] = {lo(W(t, 0)), hi(W(t, 0)), lo(W(t, 1))}, ns[3] = {hi(W(t, 1)), lo(W(t, 2)), hi(W(t, 2))};
    const int cs[3] = {lo(W(t, 3)), hi(W(t, 3)), lo(W(t, 4))};
    // the three decoded vertices must be a cyclic rotation of the triangle, neighbours rotate along
    int r = -1;
    for (int k = 0; k < 3; ++k)
      if (vs[0] == vslot[h.tri[4 * t + k]]) r = k;
    ok &= r >= 0;
    for (int k = 0; k < 3 && r >= 0; ++k) {
      ok &= vs[k] == vslot[h.tri[4 * t + (k + r) % 3]];
      ok &= ns[k] == tslot[h.tri_nbr[4 * t + (k + r) % 3]];
      ok &= cs[k] < sc.n_cslots - 8 && !seen_c[cs[k]]++;
      if (cs[k] < sc.n_cslots) corner_slots[h.tri[4 * t + (k + r) % 3]].push_back(cs[k]);
    }
  }
  // stores: quarter warps of 8 consecutive triangle threads, per pass and corner
  for (int t0q = 0; t0q < sc.tpt * sc.ttri; t0q += 8)
    for (int k = 0; k < 3; ++k) {
      int mult[8] = {0, 0, 0, 0, 0, 0, 0, 0}, w = 0;
      for (int t = t0q; t < std::min(t0q + 8, h.T); ++t) {
        const int slot = k == 0 ? lo(W(t, 3)) : (k == 1 ? hi(W(t, 3)) : lo(W(t, 4)));
        w = std::max(w, ++mult[slot % 8]);
      }
      worst_store = std::max(worst_store, double(w));
    }
  // gathers: quarter warps of 8 consecutive vertices, per read position; every vertex must read
  // exactly its own corner slots (in any order) and zero slots otherwise
  const int vwords = 1 + sc.maxv / 2;
  for (int v0 = 0; v0 < h.n; v0 += 8)
    for (int k = 0; k < sc.maxv; ++k) {
      std::vector<int> slots;
      for (int v = v0; v < std::min(v0 + 8, h.n); ++v) {
        const uint32_t w = sc.vtx_words[size_t(1 + k / 2) * sc.vstride + v];
        slots.push_back((k & 1) ? hi(w) : lo(w));
      }
      int mult[8] = {0, 0, 0, 0, 0, 0, 0, 0}, w = 0;
      for (size_t i = 0; i < slots.size(); ++i) {
        bool dup = false;
        for (size_t j = 0; j < i; ++j) dup |= slots[j] == slots[i];
        if (!dup) w = std::max(w, ++mult[slots[i] % 8]);
      }
      worst_gather = std::max(worst_gather, double(w));
    }
  for (int v = 0; v < h.n; ++v) {
    std::vector<int> reads;
    for (int k = 0; k < sc.maxv; ++k) {
      const uint32_t w = sc.vtx_words[size_t(1 + k / 2) * sc.vstride + v];
      const int slot = (k & 1) ? hi(w) : lo(w);
      if (slot < sc.n_cslots - 8) reads.push_back(slot);
      else ok &= slot < sc.n_cslots;
    }
    std::sort(reads.begin(), reads.end());
    std::sort(corner_slots[v].begin(), corner_slots[v].end());
    ok &= reads == corner_slots[v];
  }
  (void)vwords;
  stats[5] = worst_store;
  stats[6] = worst_gather;
  stats[7] = ok ? 1 : 0;
  return NPFEM_OK;
}

int npfem_quad_schedule_stats(const npfem_cell_type *type, double dt, double *stats, int32_t n_stats) {
  if (!type || !stats || n_stats < 10 || !(dt > 0)) return fail(nullptr, NPFEM_EINVAL, "type/stats missing, n_stats < 10 or dt <= 0");
  std::fill(stats, stats + n_stats, 0.0);
  HostTypeData h;
  std::string err;
  const int rc = build_host_type(*type, dt, h, err);
  if (rc != NPFEM_OK) return fail(nullptr, rc, err);
  QuadSchedule qs;
  const auto t0 = std::chrono::steady_clock::now();
  if (!build_quad_schedule(h, type->rest_positions, qs)) return NPFEM_OK;
  stats[9] = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
  stats[0] = 1;
  stats[1] = qs.threads;
  stats[2] = qs.maxq;
  stats[3] = qs.wf_vertex;
  stats[4] = qs.wf_normal;
  stats[8] = double(qs.n_vslots + qs.n_tslots + qs.n_cslots) * 16.0;
  // ---- decode the tables and check them against the mesh's own connectivity (nothing of the builder is reused) ----
  auto lo = [](uint32_t w) { return int(w & 0xffffu) / 16; };
  auto hi = [](uint32_t w) { return int(w >> 16) / 16; };
  bool ok = qs.nq * 2 == h.T;
  std::vector<int> vertex_of_slot(size_t(qs.n_vslots), -1);
  for (int v = 0; v < h.n; ++v) {
    const int sl = lo(qs.vtx_words[v]);
    ok &= sl < qs.n_vslots && vertex_of_slot[sl] < 0;
    if (sl < qs.n_vslots) vertex_of_slot[sl] = v;
  }
  // directed edge (a, b) -> the triangle that runs a -> b (closed oriented manifold: exactly one)
  std::vector<int> tri_of_edge(size_t(h.n) * h.n, -1);
  for (int t = 0; t < h.T; ++t)
    for (int k = 0; k < 3; ++k) tri_of_edge[size_t(h.tri[4 * t + k]) * h.n + h.tri[4 * t + (k + 1) % 3]] = t;
  auto tri_at = [&](int a, int b) { return a >= 0 && b >= 0 ? tri_of_edge[size_t(a) * h.n + b] : -1; };
  auto W = [&](int k, int q) { return qs.quad_words[size_t(q) * qs.threads + k]; };
  std::vector<int> quad_of_tri(size_t(h.T), -1), tslot_of_tri(size_t(h.T), -1), seen_t(size_t(qs.n_tslots), 0),
      seen_c(size_t(qs.n_cslots), 0);
  std::vector<std::vector<int>> corner_slots(size_t(h.n));
  struct Dec { int p, q, r, s, A, B; };
  std::vector<Dec> dec(size_t(qs.nq), Dec{-1, -1, -1, -1, -1, -1});
  for (int k = 0; k < qs.nq && ok; ++k) {
    const int sl[4] = {lo(W(k, 0)), hi(W(k, 0)), lo(W(k, 1)), hi(W(k, 1))};
    int v[4];
    for (int i = 0; i < 4; ++i) v[i] = sl[i] < qs.n_vslots ? vertex_of_slot[sl[i]] : -1;
    Dec &d = dec[k];
    d.p = v[0]; d.q = v[1]; d.r = v[2]; d.s = v[3];
    d.A = tri_at(d.p, d.q);                     // T0 = (p, q, r)
    d.B = tri_at(d.q, d.p);                     // T1 = (p, s, q)
    ok &= d.A >= 0 && d.B >= 0 && d.A != d.B && tri_at(d.q, d.r) == d.A && tri_at(d.r, d.p) == d.A &&
          tri_at(d.p, d.s) == d.B && tri_at(d.s, d.q) == d.B;
    if (!ok) break;
    ok &= quad_of_tri[d.A] < 0 && quad_of_tri[d.B] < 0;
    quad_of_tri[d.A] = quad_of_tri[d.B] = k;
    const int ta = lo(W(k, 4)), tb = hi(W(k, 4));
    ok &= ta < qs.n_tslots && tb < qs.n_tslots && ta != tb && !seen_t[ta]++ && !seen_t[tb]++;
    tslot_of_tri[d.A] = ta;
    tslot_of_tri[d.B] = tb;
    const int cs[4] = {lo(W(k, 5)), hi(W(k, 5)), lo(W(k, 6)), hi(W(k, 6))};
    for (int i = 0; i < 4; ++i) {
      ok &= cs[i] < qs.n_cslots - 8 && !seen_c[cs[i]]++;
      corner_slots[v[i]].push_back(cs[i]);
    }
  }
  for (int t = 0; t < h.T; ++t) ok &= quad_of_tri[t] >= 0;
  // neighbour normals across the four outer edges q-r, r-p (of T0), p-s, s-q (of T1)
  for (int k = 0; k < qs.nq && ok; ++k) {
    const Dec &d = dec[k];
    const int ns[4] = {lo(W(k, 2)), hi(W(k, 2)), lo(W(k, 3)), hi(W(k, 3))};
    const int nb[4] = {tri_at(d.r, d.q), tri_at(d.p, d.r), tri_at(d.s, d.p), tri_at(d.q, d.s)};
    for (int i = 0; i < 4; ++i) ok &= nb[i] >= 0 && ns[i] == tslot_of_tri[nb[i]];
  }
  // stores: quarter warps of 8 consecutive quad threads, per corner role (one STS.128 each)
  double worst_store = 0, worst_gather = 0;
  for (int k0 = 0; k0 < qs.nq; k0 += 8)
    for (int role = 0; role < 4; ++role) {
      int mult[8] = {0, 0, 0, 0, 0, 0, 0, 0}, w = 0;
      for (int k = k0; k < std::min(k0 + 8, qs.nq); ++k) {
        const uint32_t word = W(k, 5 + role / 2);
        w = std::max(w, ++mult[((role & 1) ? hi(word) : lo(word)) % 8]);
      }
      worst_store = std::max(worst_store, double(w));
    }
  // gathers: quarter warps of 8 consecutive vertices, per read position; a vertex reads exactly the slots its quads
  // write for it (any order) and zero slots otherwise
  auto read_slot = [&](int v, int k) {
    const uint32_t w = qs.vtx_words[size_t(1 + k / 2) * qs.vstride + v];
    return (k & 1) ? hi(w) : lo(w);
  };
  for (int v0 = 0; v0 < h.n; v0 += 8)
    for (int k = 0; k < qs.maxq; ++k) {
      int mult[8] = {0, 0, 0, 0, 0, 0, 0, 0}, w = 0;
      std::vector<int> slots;
      for (int v = v0; v < std::min(v0 + 8, h.n); ++v) {
        const int sl = read_slot(v, k);
        if (std::find(slots.begin(), slots.end(), sl) == slots.end()) w = std::max(w, ++mult[sl % 8]);
        slots.push_back(sl);
      }
      worst_gather = std::max(worst_gather, double(w));
    }
  for (int v = 0; v < h.n; ++v) {
    std::vector<int> reads;
    for (int k = 0; k < qs.maxq; ++k) {
      const int sl = read_slot(v, k);
      if (sl < qs.n_cslots - 8) reads.push_back(sl);
      else ok &= sl < qs.n_cslots;
    }
    std::sort(reads.begin(), reads.end());
    std::sort(corner_slots[v].begin(), corner_slots[v].end());
    ok &= reads == corner_slots[v];
  }
  stats[5] = worst_store;
  stats[6] = worst_gather;
  stats[7] = ok ? 1 : 0;
  return NPFEM_OK;
}

int npfem_quadmp_schedule_stats(const npfem_cell_type *type, double dt, double *stats, int32_t n_stats) {
  if (!type || !stats || n_stats < 10 || !(dt > 0)) return fail(nullptr, NPFEM_EINVAL, "type/stats missing, n_stats < 10 or dt <= 0");
  std::fill(stats, stats + n_stats, 0.0);
  HostTypeData h;
  std::string err;
  const int rc = build_host_type(*type, dt, h, err);
  if (rc != NPFEM_OK) return fail(nullptr, rc, err);
  QuadMpSchedule qs;
  const auto t0 = std::chrono::steady_clock::now();
  if (!build_quadmp_schedule(h, type->rest_positions, qs)) return NPFEM_OK;
  stats[9] = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
  stats[0] = 1;
  stats[1] = qs.passes;
  stats[2] = qs.maxq;
  stats[3] = qs.wf_vertex;
  stats[4] = qs.wf_normal;
  stats[8] = double(qs.n_vslots + qs.n_tslots + qs.n_cslots) * 16.0 + 12.0 * ((h.n + 15) / 16 * 16);
  // ---- decode the tables and check them against the mesh's own connectivity ---------------------------------------
  auto lo = [](uint32_t w) { return int(w & 0xffffu); };
  auto hi = [](uint32_t w) { return int(w >> 16); };
  const int TH = qs.threads, vwords = 1 + qs.maxq / 2;
  bool ok = qs.nq * 2 == h.T && qs.passes * TH >= qs.nq;
  std::vector<int> vertex_of_slot(size_t(qs.n_vslots), -1);
  for (int v = 0; v < h.n; ++v) {
    const int sl = int(qs.vtx_slot[v]);
    ok &= sl < qs.n_vslots && vertex_of_slot[sl] < 0;
    if (sl < qs.n_vslots) vertex_of_slot[sl] = v;
  }
  std::vector<int> tri_of_edge(size_t(h.n) * h.n, -1);
  for (int t = 0; t < h.T; ++t)
    for (int k = 0; k < 3; ++k) tri_of_edge[size_t(h.tri[4 * t + k]) * h.n + h.tri[4 * t + (k + 1) % 3]] = t;
  auto tri_at = [&](int a, int b) { return a >= 0 && b >= 0 ? tri_of_edge[size_t(a) * h.n + b] : -1; };
  auto W = [&](int k, int q) { return qs.quad_words[(size_t(k / TH) * 7 + q) * TH + k % TH]; };
  std::vector<int> quad_of_tri(size_t(h.T), -1), tslot_of_tri(size_t(h.T), -1), seen_t(size_t(qs.n_tslots), 0);
  struct Dec { int p, q, r, s, A, B; };
  std::vector<Dec> dec(size_t(qs.nq), Dec{-1, -1, -1, -1, -1, -1});
  double worst_store = 0, worst_gather = 0;
  for (int ps = 0; ps < qs.passes && ok; ++ps) {
    const int k0 = ps * TH, k1 = std::min(qs.nq, k0 + TH);
    std::vector<int> seen_c(size_t(qs.n_cslots), 0);
    std::vector<std::vector<int>> corner_slots(size_t(h.n));
    for (int k = k0; k < k1 && ok; ++k) {
      const int sl[4] = {lo(W(k, 0)), hi(W(k, 0)), lo(W(k, 1)), hi(W(k, 1))};
      int v[4];
      for (int i = 0; i < 4; ++i) v[i] = sl[i] < qs.n_vslots ? vertex_of_slot[sl[i]] : -1;
      Dec &d = dec[k];
      d.p = v[0]; d.q = v[1]; d.r = v[2]; d.s = v[3];
      d.A = tri_at(d.p, d.q);
      d.B = tri_at(d.q, d.p);
      ok &= d.A >= 0 && d.B >= 0 && d.A != d.B && tri_at(d.q, d.r) == d.A && tri_at(d.r, d.p) == d.A &&
            tri_at(d.p, d.s) == d.B && tri_at(d.s, d.q) == d.B;
      if (!ok) break;
      ok &= quad_of_tri[d.A] < 0 && quad_of_tri[d.B] < 0;
      quad_of_tri[d.A] = quad_of_tri[d.B] = k;
      const int ta = lo(W(k, 4)), tb = hi(W(k, 4));
      ok &= ta < qs.n_tslots && tb < qs.n_tslots && ta != tb && !seen_t[ta]++ && !seen_t[tb]++;
      tslot_of_tri[d.A] = ta;
      tslot_of_tri[d.B] = tb;
      const int cs[4] = {lo(W(k, 5)), hi(W(k, 5)), lo(W(k, 6)), hi(W(k, 6))};
      for (int i = 0; i < 4; ++i) {
        ok &= cs[i] < qs.n_cslots - 8 && !seen_c[cs[i]]++;
        corner_slots[v[i]].push_back(cs[i]);
      }
    }
    // stores: quarter warps of 8 consecutive quad threads, per corner role
    for (int k = k0; k < k1; k += 8)
      for (int role = 0; role < 4; ++role) {
        int mult[8] = {0, 0, 0, 0, 0, 0, 0, 0}, w = 0;
        for (int kk = k; kk < std::min(k + 8, k1); ++kk) {
          const uint32_t word = W(kk, 5 + role / 2);
          w = std::max(w, ++mult[((role & 1) ? hi(word) : lo(word)) % 8]);
        }
        worst_store = std::max(worst_store, double(w));
      }
    // the pass's vertex list: every vertex touched by the pass exactly once, reading exactly its slots
    const int len = qs.list_len[ps];
    ok &= len <= qs.lstride;
    auto LW = [&](int q, int e) { return qs.list_words[(size_t(ps) * vwords + q) * qs.lstride + e]; };
    auto read_slot = [&](int e, int q) { const uint32_t w = LW(1 + q / 2, e); return (q & 1) ? hi(w) : lo(w); };
    std::vector<int> listed(size_t(h.n), 0);
    for (int e = 0; e < len && ok; ++e) {
      const int v = int(LW(0, e));
      ok &= v >= 0 && v < h.n && !listed[v]++;
      if (!ok) break;
      std::vector<int> reads;
      for (int q = 0; q < qs.maxq; ++q) {
        const int sl = read_slot(e, q);
        if (sl < qs.n_cslots - 8) reads.push_back(sl);
        else ok &= sl < qs.n_cslots;
      }
      std::sort(reads.begin(), reads.end());
      std::sort(corner_slots[v].begin(), corner_slots[v].end());
      ok &= reads == corner_slots[v];
    }
    for (int e = len; e < qs.lstride; ++e) ok &= LW(0, e) == 0xffffffffu;
    for (int v = 0; v < h.n; ++v) ok &= listed[v] || corner_slots[v].empty();
    for (int e0 = 0; e0 < len; e0 += 8)
      for (int q = 0; q < qs.maxq; ++q) {
        int mult[8] = {0, 0, 0, 0, 0, 0, 0, 0}, w = 0;
        std::vector<int> slots;
        for (int e = e0; e < std::min(e0 + 8, len); ++e) {
          const int sl = read_slot(e, q);
          if (std::find(slots.begin(), slots.end(), sl) == slots.end()) w = std::max(w, ++mult[sl % 8]);
          slots.push_back(sl);
        }
        worst_gather = std::max(worst_gather, double(w));
      }
  }
  for (int t = 0; t < h.T; ++t) ok &= quad_of_tri[t] >= 0;
  for (int k = 0; k < qs.nq && ok; ++k) {
    const Dec &d = dec[k];
    const int ns[4] = {lo(W(k, 2)), hi(W(k, 2)), lo(W(k, 3)), hi(W(k, 3))};
    const int nb[4] = {tri_at(d.r, d.q), tri_at(d.p, d.r), tri_at(d.s, d.p), tri_at(d.q, d.s)};
    for (int i = 0; i < 4; ++i) ok &= nb[i] >= 0 && ns[i] == tslot_of_tri[nb[i]];
  }
  stats[5] = worst_store;
  stats[6] = worst_gather;
  stats[7] = ok ? 1 : 0;
  return NPFEM_OK;
}

void npfem_destroy(npfem_ctx *c) {
  if (!c) return;
  cudaSetDevice(c->device);
  cudaStreamSynchronize(c->stream);
  if (c->ws_owned && c->ws) cudaFree(c->ws);
  for (auto &m : c->feat)
    if (m.owned && m.base) cudaFree(m.base);
  for (auto &sp : c->spans) {
    cudaEventDestroy(sp.a);
    cudaEventDestroy(sp.b);
  }
  for (auto e : c->event_pool) cudaEventDestroy(e);
  for (auto e : c->io_events) cudaEventDestroy(e);
  if (c->h2d_stream) cudaStreamDestroy(c->h2d_stream);
  if (c->d2h_stream) cudaStreamDestroy(c->d2h_stream);
  cudaGetLastError();
  delete c;
}

}  // extern "C"
