// Create-time schedule of the MULTI-PASS quad local step (local_quadmp.cu): see quad_schedule.hpp for the pairing and
// the colouring; this file only differs in how the result is laid out (passes of 640 quads, per-pass corner slots).
#pragma once
#include "quad_schedule.hpp"

namespace npfem {

// Multi-pass variant of the quad schedule (quadmp_schedule.hpp is included after quad_schedule.hpp): the quads of a
// large mesh in PASSES of QMP_THREADS, one quad per thread and pass; vertex / normal slots are global to the cell,
// corner-force slots and the lists of vertices that gather them are per pass.
constexpr int QMP_THREADS = 640, QMP_MAX_PASSES = 4;

struct QuadMpSchedule {
  bool valid = false;
  int threads = 0, passes = 0, nq = 0, maxq = 0;
  int n_vslots = 0, n_tslots = 0, n_cslots = 0;   // float4 slots of sx / sN (whole cell) and of sC (one pass)
  int lstride = 0;                                 // row stride of the per-pass vertex lists (<= 2 * threads)
  std::vector<uint32_t> quad_words;    // [passes][7][threads] packed 16-bit slot INDICES (see local_quadmp.cu)
  std::vector<float> quad_consts;      // [passes][22][threads]
  std::vector<uint32_t> list_words;    // [passes][1 + maxq/2][lstride]: vertex id (0xffffffff = none), corner slots
  std::vector<int> list_len;           // [passes]
  std::vector<uint32_t> vtx_slot;      // [n rounded up to 32] slot of the vertex in sx
  std::vector<float> vtx_coef;         // [n rounded up to 32]
  std::vector<int> mate;
  double wf_vertex = 0, wf_normal = 0;
  double vol_lane_bound = 0;
  int quads_at_vertex_max = 0;
  double quads_at_vertex_mean = 0;
};

// Builds the multi-pass quad schedule of one cell type (meshes too large for one pass of 640 quads: RBC-2562 has 2,560).
// X = rest positions [n][3].  Returns false (valid stays false) when the type does not fit (odd triangle count, no
// perfect matching, more than QMP_MAX_PASSES passes, slot arrays beyond the 16-bit indices of the tables).
inline bool build_quadmp_schedule(const HostTypeData &h, const double *X, QuadMpSchedule &out, int repair_rounds = 24) {
  using namespace sched_detail;
  using namespace quad_detail;
  out = QuadMpSchedule();
  const int n = h.n, T = h.T;
  if (h.valence_max > 8 || (T & 1)) return false;
  const int nq = T / 2;
  const int threads = QMP_THREADS;
  const int passes = (nq + threads - 1) / threads;
  if (passes < 1 || passes > QMP_MAX_PASSES) return false;
  const int qthreads = passes * threads;            // quad k = pass k / threads, thread k % threads
  const int n_vslots = (n + 7) / 8 * 8, n_tslots = 2 * qthreads;
  const int octs_q = threads / 8;                   // write octets of ONE pass
  const int n_wgroups = 4 * octs_q;                 // corner-force write groups (role, octet) of one pass
  const int n_cslots = 8 * n_wgroups + 8;           // per pass; + 8 zero slots, one per bank group
  if (n_vslots > 65535 || n_tslots > 65535) return false;

  // ---- matching ------------------------------------------------------------------------------
  std::vector<std::array<int, 3>> adj(static_cast<size_t>(T));
  for (int t = 0; t < T; ++t) adj[t] = {h.tri_nbr[4 * t], h.tri_nbr[4 * t + 1], h.tri_nbr[4 * t + 2]};
  Blossom bl(T, adj);
  if (bl.solve() != nq) return false;
  std::vector<int> mate = bl.match;
  repair_matching(h, adj, mate, repair_rounds);
  out.mate = mate;
  {
    const std::vector<int> cnt = quads_at_vertices(h, mate);
    long sum = 0;
    for (int c : cnt) { out.quads_at_vertex_max = std::max(out.quads_at_vertex_max, c); sum += c; }
    out.quads_at_vertex_mean = double(sum) / n;
  }
  const int maxq = out.quads_at_vertex_max <= 6 ? 6 : 8;     // reads per vertex of the kernel's variants

  // ---- quads in order of their smaller triangle; (A, B) = (smaller, larger) before the swap search --------------
  std::vector<int> qa, qb;                          // quad -> its two triangles
  for (int t = 0; t < T; ++t)
    if (mate[t] > t) { qa.push_back(t); qb.push_back(mate[t]); }
  if (int(qa.size()) != nq) return false;
  std::vector<int> swp(static_cast<size_t>(nq), 0);
  struct Roles { int p, q, r, s, n0, n1, n2, n3, A, sA, B, sB; };
  auto roles = [&](int k) {
    const int A = swp[k] ? qb[k] : qa[k], B = swp[k] ? qa[k] : qb[k];
    int sA = -1, sB = -1;
    for (int s = 0; s < 3; ++s) {
      if (h.tri_nbr[4 * A + s] == B) sA = s;
      if (h.tri_nbr[4 * B + s] == A) sB = s;
    }
    Roles R{};
    R.A = A; R.B = B; R.sA = sA; R.sB = sB;
    R.p = h.tri[4 * A + sA]; R.q = h.tri[4 * A + (sA + 1) % 3]; R.r = h.tri[4 * A + (sA + 2) % 3];
    R.s = h.tri[4 * B + (sB + 2) % 3];
    R.n0 = h.tri_nbr[4 * A + (sA + 1) % 3];        // T0 across q-r
    R.n1 = h.tri_nbr[4 * A + (sA + 2) % 3];        // T0 across r-p
    R.n2 = h.tri_nbr[4 * B + (sB + 1) % 3];        // T1 = (p, s, q) across p-s
    R.n3 = h.tri_nbr[4 * B + (sB + 2) % 3];        // T1 across s-q
    return R;
  };
  // a triangle's index for the normal slots: T0 of quad k -> k, T1 of quad k -> qthreads + k
  std::vector<int> quad_of(static_cast<size_t>(T));
  for (int k = 0; k < nq; ++k) { quad_of[qa[k]] = k; quad_of[qb[k]] = k; }
  auto tau = [&](int t) {
    const int k = quad_of[t];
    const bool first = (swp[k] ? qb[k] : qa[k]) == t;
    return first ? k : qthreads + k;
  };

  OctetColouring vc, tc;
  vc.init(n);
  tc.init(n_tslots);
  Lcg rng(uint64_t(n) * 40503u + uint64_t(T));
  auto build_groups = [&]() {
    std::vector<std::array<int, 8>> vg, ng;
    for (int role = 0; role < 4; ++role)
      for (int o = 0; o < qthreads; o += 8) {
        std::array<int, 8> a, b;
        for (int i = 0; i < 8; ++i) {
          const int k = o + i;
          if (k >= nq) { a[i] = b[i] = -1; continue; }
          const Roles R = roles(k);
          a[i] = role == 0 ? R.p : (role == 1 ? R.q : (role == 2 ? R.r : R.s));
          b[i] = tau(role == 0 ? R.n0 : (role == 1 ? R.n1 : (role == 2 ? R.n2 : R.n3)));
        }
        vg.push_back(a);
        ng.push_back(b);
      }
    vc.set_groups(vg);
    tc.set_groups(ng);
  };
  const int rounds = 6, sweeps = 10;
  for (int r = 0; r < rounds; ++r) {
    build_groups();
    for (int s = 0; s < sweeps; ++s) { vc.sweep(rng); tc.sweep(rng); }
    // best (T0, T1) order of the 8 quads of every octet, colours fixed (2^8 combinations).  Swapping a quad changes
    // which normal slot (k or qthreads + k) each of its triangles owns, hence what OTHER quads' neighbour gathers read;
    // that second-order effect is picked up by the next round's sweeps.
    for (int o = 0; o < qthreads; o += 8) {
      const int cnt = std::min(8, nq - o);
      if (cnt <= 0) continue;
      int best_cost = 1 << 30, best_combo = 0;
      int keep[8];
      for (int i = 0; i < cnt; ++i) keep[i] = swp[o + i];
      for (int combo = 0; combo < (1 << cnt); ++combo) {
        for (int i = 0; i < cnt; ++i) swp[o + i] = (combo >> i) & 1;
        int cost = 0;
        for (int role = 0; role < 4 && cost < best_cost; ++role) {
          int vi[8], ti[8];
          for (int i = 0; i < cnt; ++i) {
            const Roles R = roles(o + i);
            vi[i] = role == 0 ? R.p : (role == 1 ? R.q : (role == 2 ? R.r : R.s));
            ti[i] = tau(role == 0 ? R.n0 : (role == 1 ? R.n1 : (role == 2 ? R.n2 : R.n3)));
          }
          cost += group_cost(vi, cnt, vc.colour) + group_cost(ti, cnt, tc.colour);
        }
        if (cost < best_cost) { best_cost = cost; best_combo = combo; }
      }
      for (int i = 0; i < cnt; ++i) swp[o + i] = (best_combo >> i) & 1;
      (void)keep;
    }
  }
  build_groups();
  for (int s = 0; s < sweeps; ++s) { vc.sweep(rng); tc.sweep(rng); }
  out.wf_vertex = 4.0 * double(vc.total()) / double(vc.groups.size());
  out.wf_normal = 4.0 * double(tc.total()) / double(tc.groups.size());
  auto vslot = [&](int v) { return 8 * (v / 8) + vc.colour[v]; };
  auto tslot = [&](int t) { const int x = tau(t); return 8 * (x / 8) + tc.colour[x]; };

  // ---- per pass: the vertices its quads touch (list entries), corner-force slots by exact bipartite edge colouring
  //      ({write groups of the pass} x {read groups = octets of list entries}, degree <= 8) --------------------------
  out.threads = threads; out.passes = passes; out.nq = nq; out.maxq = maxq;
  out.n_vslots = n_vslots; out.n_tslots = n_tslots; out.n_cslots = n_cslots;
  const int vwords = 1 + maxq / 2;
  std::vector<std::vector<int>> list(static_cast<size_t>(passes));            // pass -> vertices in entry order
  std::vector<std::vector<std::array<int, 8>>> reads(static_cast<size_t>(passes));
  std::vector<int> cslot_of(size_t(nq) * 4, -1);
  int lstride = 0;
  for (int ps = 0; ps < passes; ++ps) {
    const int k0 = ps * threads, k1 = std::min(nq, k0 + threads);
    std::vector<int> entry(static_cast<size_t>(n), -1);
    std::vector<int> &L = list[ps];
    for (int k = k0; k < k1; ++k) {
      const Roles R = roles(k);
      const int vs[4] = {R.p, R.q, R.r, R.s};
      for (int v : vs)
        if (entry[v] < 0) { entry[v] = int(L.size()); L.push_back(v); }
    }
    const int octs_l = (int(L.size()) + 7) / 8;
    std::vector<int> fill(L.size(), 0);
    std::vector<int> read_pos(size_t(k1 - k0) * 4);
    std::vector<std::pair<int, int>> edges(size_t(k1 - k0) * 4);
    for (int k = k0; k < k1; ++k) {
      const Roles R = roles(k);
      const int vs[4] = {R.p, R.q, R.r, R.s};
      for (int role = 0; role < 4; ++role) {
        const int e = entry[vs[role]], pos = fill[e]++;
        if (pos >= maxq) return false;
        read_pos[4 * (k - k0) + role] = pos;
        edges[4 * (k - k0) + role] = {role * octs_q + (k - k0) / 8, pos * octs_l + e / 8};
      }
    }
    const std::vector<int> ecol = bipartite_edge_colouring8(n_wgroups, maxq * octs_l, edges);
    if (ecol.size() != edges.size()) return false;
    reads[ps].assign(L.size(), std::array<int, 8>());
    for (auto &r : reads[ps]) r.fill(-1);
    for (int k = k0; k < k1; ++k) {
      const Roles R = roles(k);
      const int vs[4] = {R.p, R.q, R.r, R.s};
      for (int role = 0; role < 4; ++role) {
        const int cs = 8 * edges[4 * (k - k0) + role].first + ecol[4 * (k - k0) + role];
        cslot_of[4 * k + role] = cs;
        reads[ps][entry[vs[role]]][read_pos[4 * (k - k0) + role]] = cs;
      }
    }
    // padding reads: zero slots of a bank group the read group does not use
    for (int q = 0; q < maxq; ++q)
      for (int o = 0; o < int(L.size()); o += 8) {
        bool used[8] = {false, false, false, false, false, false, false, false};
        for (int e = o; e < std::min(o + 8, int(L.size())); ++e)
          if (reads[ps][e][q] >= 0) used[reads[ps][e][q] % 8] = true;
        int free_colour = 0;
        while (free_colour < 7 && used[free_colour]) ++free_colour;
        for (int e = o; e < std::min(o + 8, int(L.size())); ++e)
          if (reads[ps][e][q] < 0) reads[ps][e][q] = 8 * n_wgroups + free_colour;
      }
    lstride = std::max(lstride, (int(L.size()) + 31) / 32 * 32);
  }
  if (lstride > 2 * threads) return false;            // a thread handles at most two list entries per pass
  out.lstride = lstride;

  // ---- tables (slot INDICES, 16 bit each; the kernel scales them by 16 bytes) ---------------------------------
  out.quad_words.assign(size_t(passes) * 7 * threads, 0u);
  out.quad_consts.assign(size_t(passes) * 22 * threads, 0.f);
  out.list_words.assign(size_t(passes) * vwords * lstride, 0u);
  out.list_len.assign(static_cast<size_t>(passes), 0);
  out.vtx_slot.assign(size_t((n + 31) / 32 * 32), 0u);
  out.vtx_coef.assign(size_t((n + 31) / 32 * 32), 0.f);
  const npfem_material &m = h.mat;
  const double B4 = m.skalak_B / 4.0, C4 = m.skalak_C / 4.0;
  // rest metric of a triangle with corners (x0, x1, x2): R = Dm^-1 Dm^-T, J = det(Dm^-1)^2, A0 (reading R5)
  auto metric = [&](int v0, int v1, int v2, float *K) {
    const double *x0 = X + 3 * v0, *x1 = X + 3 * v1, *x2 = X + 3 * v2;
    double E1[3], E2[3], N[3];
    for (int q = 0; q < 3; ++q) { E1[q] = x1[q] - x0[q]; E2[q] = x2[q] - x0[q]; }
    cross3(E1, E2, N);
    const double len1 = std::sqrt(dot3(E1, E1)), twoA = std::sqrt(dot3(N, N));
    const double a = 1.0 / len1, height = twoA / len1, c = 1.0 / height;
    const double b = -(dot3(E2, E1) / len1) / (len1 * height), A0 = 0.5 * twoA;
    const double J = (a * c) * (a * c);
    K[0] = float(a * a + b * b); K[1] = float(b * c); K[2] = float(c * c); K[3] = float(J);
    K[4] = float(2.0 * A0 * B4); K[5] = float(2.0 * A0 * J * C4);
    return A0;
  };
  double cen[3] = {0, 0, 0}, rmax = 0;
  for (int v = 0; v < n; ++v)
    for (int q = 0; q < 3; ++q) cen[q] += X[3 * v + q] / n;
  for (int v = 0; v < n; ++v) {
    double r2 = 0;
    for (int q = 0; q < 3; ++q) r2 += (X[3 * v + q] - cen[q]) * (X[3 * v + q] - cen[q]);
    rmax = std::max(rmax, std::sqrt(r2));
  }
  std::vector<double> lane_bound(static_cast<size_t>(threads), 0.0);
  for (int k = 0; k < nq; ++k) {
    const Roles R = roles(k);
    const int ps = k / threads, t = k % threads;
    auto W = [&](int q) -> uint32_t & { return out.quad_words[(size_t(ps) * 7 + q) * threads + t]; };
    auto K = [&](int q) -> float & { return out.quad_consts[(size_t(ps) * 22 + q) * threads + t]; };
    W(0) = uint32_t(vslot(R.p)) | uint32_t(vslot(R.q)) << 16;
    W(1) = uint32_t(vslot(R.r)) | uint32_t(vslot(R.s)) << 16;
    W(2) = uint32_t(tslot(R.n0)) | uint32_t(tslot(R.n1)) << 16;
    W(3) = uint32_t(tslot(R.n2)) | uint32_t(tslot(R.n3)) << 16;
    W(4) = uint32_t(tslot(R.A)) | uint32_t(tslot(R.B)) << 16;
    W(5) = uint32_t(cslot_of[4 * k + 0]) | uint32_t(cslot_of[4 * k + 1]) << 16;
    W(6) = uint32_t(cslot_of[4 * k + 2]) | uint32_t(cslot_of[4 * k + 3]) << 16;
    float K0[6], K1[6];
    const double A0 = metric(R.p, R.q, R.r, K0);     // T0 = (p, q, r)
    const double A1 = metric(R.p, R.s, R.q, K1);     // T1 = (p, s, q)
    for (int q = 0; q < 6; ++q) { K(q) = K0[q]; K(6 + q) = K1[q]; }
    // hinge rest angles belong to the edges: shared p-q (side sA of A), q-r, r-p of A, p-s, s-q of B
    const int hs[5][2] = {{R.A, R.sA}, {R.A, (R.sA + 1) % 3}, {R.A, (R.sA + 2) % 3}, {R.B, (R.sB + 1) % 3}, {R.B, (R.sB + 2) % 3}};
    for (int e = 0; e < 5; ++e) {
      K(12 + e) = float(m.k_bending * h.hinge_rest[6 * hs[e][0] + 2 * hs[e][1] + 0]);
      K(17 + e) = float(m.k_bending * h.hinge_rest[6 * hs[e][0] + 2 * hs[e][1] + 1]);
    }
    lane_bound[t] += rmax * 2.0 * (A0 + A1);          // a lane sums its quads of all passes before the REDUX
  }
  for (double b : lane_bound) out.vol_lane_bound = std::max(out.vol_lane_bound, b);
  for (int ps = 0; ps < passes; ++ps) {
    out.list_len[ps] = int(list[ps].size());
    for (int e = 0; e < int(list[ps].size()); ++e) {
      out.list_words[(size_t(ps) * vwords) * lstride + e] = uint32_t(list[ps][e]);
      for (int q = 0; q < maxq / 2; ++q)
        out.list_words[(size_t(ps) * vwords + 1 + q) * lstride + e] =
            uint32_t(reads[ps][e][2 * q]) | (uint32_t(reads[ps][e][2 * q + 1]) << 16);
    }
    for (int e = int(list[ps].size()); e < lstride; ++e)
      out.list_words[(size_t(ps) * vwords) * lstride + e] = 0xffffffffu;      // no vertex
  }
  const double gamma = (m.rayleigh_beta / h.h) / (1.0 + m.rayleigh_beta / h.h);
  const double inertia = (1.0 + h.h * m.rayleigh_alpha) / (h.h * h.h);
  for (int v = 0; v < n; ++v) {
    out.vtx_slot[v] = uint32_t(vslot(v));
    out.vtx_coef[v] = float((1.0 - gamma) * inertia * h.mass[v]);
  }
  out.valid = true;
  return true;
}

}  // namespace npfem
