// Create-time "schedule" of the fp32 scheduled local step (local_sched.cu): which thread owns
// which triangles / vertex, and WHERE in shared memory every vertex position, triangle normal and
// corner force lives, chosen so that the three gathers of the kernel are (nearly) free of
// shared-memory bank conflicts.
//
// Why: a 128-bit shared load is served 8 lanes (a quarter warp) per wavefront; the 8 lanes hit
// distinct banks only if their 16-byte slot numbers are distinct modulo 8.  With the mesh's own
// vertex / triangle / corner numbering the gathers cost 6-13 wavefronts instead of 4
// (profiles/r1_ncu_full_v3.md) and shared-memory bandwidth bound the local step.  Here
//   * vertex v    -> slot 8*(v/8) + colour_v(v)   (a permutation inside each aligned octet, so
//   * triangle t  -> slot 8*(t/8) + colour_t(t)    the owner's own store is conflict-free)
//     with the colours found by a min-conflicts search over the octets (8 consecutive
//     triangles = one quarter warp) that read them, jointly with a cyclic rotation of every
//     triangle's corner order (which gather instruction reads which corner / neighbour);
//   * corner force (t,c) -> slot 8*writegroup + colour, the colours being a proper 8-edge-colouring
//     of the bipartite multigraph {write quarter-warps} x {read quarter-warps} (maximum degree 8,
//     so Koenig's theorem guarantees one): stores AND gathers are exactly conflict-free.
// Everything here is integer / fp64 host work done once per cell TYPE (cells of a
// type share the mesh).  Product code: shares nothing with oracle/.
#pragma once

#include <algorithm>
#include <array>
#include <cmath>
#include <cstdint>
#include <vector>

#include "host_setup.hpp"

namespace npfem {

struct LocalSchedule {
  bool valid = false;
  int threads = 0;   // CTA size (multiple of 32); vertex v < threads is owned by thread v, the rest by the last warp
  int vstride = 0;   // row stride of the vertex tables (>= n)
  int tpt = 0;       // triangles per thread
  int ttri = 0;      // threads that own triangles (multiple of 8): triangle t = j*ttri + tid
  int maxv = 0;      // corner-force reads per vertex (6 or 8)
  int n_vslots = 0, n_tslots = 0, n_cslots = 0;   // float4 slots of sx / sN / sC
  std::vector<uint32_t> tri_words;   // [tpt][5][threads] packed 16-bit byte offsets (see local_sched.cu)
  std::vector<float> tri_consts;     // [tpt][12][threads] R11 R12 R22 J tA tC kc0[3] ks0[3]
  std::vector<uint32_t> vtx_words;   // [1 + maxv/2][vstride] own slot, corner-force slots
  std::vector<float> vtx_coef;       // [vstride]
  double wf_vertex = 0, wf_normal = 0;   // predicted wavefronts per gather instruction (ideal 4)
  double vol_lane_bound = 0;             // max over threads of sum_j |x_0 - centroid| 2 A_t (rest shape)
};

namespace sched_detail {

struct Lcg {   // deterministic, platform-independent
  uint64_t s;
  explicit Lcg(uint64_t seed) : s(seed * 2862933555777941757ULL + 3037000493ULL) {}
  uint32_t next() {
    s = s * 6364136223846793005ULL + 1442695040888963407ULL;
    return uint32_t(s >> 33);
  }
};

// wavefronts of one quarter-warp reading `items` (distinct items count once: broadcast)
inline int group_cost(const int *items, int cnt, const std::vector<int> &colour) {
  int mult[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  int best = 0;
  for (int i = 0; i < cnt; ++i) {
    const int it = items[i];
    if (it < 0) continue;
    bool dup = false;
    for (int k = 0; k < i; ++k) dup |= items[k] == it;
    if (dup) continue;
    const int m = ++mult[colour[it]];
    best = m > best ? m : best;
  }
  return best;
}

// items coloured by a permutation inside each aligned octet; groups = quarter-warp reads
struct OctetColouring {
  int n_items = 0, n8 = 0;
  std::vector<int> colour;                    // [n8] (entries >= n_items are placeholders)
  std::vector<std::array<int, 8>> groups;     // item ids, -1 = none
  std::vector<std::vector<int>> member;       // groups of each item
  std::vector<int> cost;

  void init(int n) {
    n_items = n;
    n8 = (n + 7) / 8 * 8;
    colour.resize(size_t(n8));
    for (int i = 0; i < n8; ++i) colour[i] = i % 8;
  }
  void set_groups(const std::vector<std::array<int, 8>> &g) {
    groups = g;
    member.assign(size_t(n8), {});
    cost.resize(groups.size());
    for (size_t gi = 0; gi < groups.size(); ++gi) {
      for (int k = 0; k < 8; ++k) {
        const int it = groups[gi][k];
        if (it < 0) continue;
        auto &m = member[it];
        if (std::find(m.begin(), m.end(), int(gi)) == m.end()) m.push_back(int(gi));
      }
      cost[gi] = group_cost(groups[gi].data(), 8, colour);
    }
  }
  long total() const {
    long t = 0;
    for (int c : cost) t += c;
    return t;
  }
  // one pass of pairwise colour swaps inside every octet; keeps a swap if it does not hurt
  void sweep(Lcg &rng) {
    std::vector<int> touched;
    for (int o = 0; o < n8; o += 8)
      for (int a = o; a < o + 8; ++a)
        for (int b = a + 1; b < o + 8; ++b) {
          if (a >= n_items && b >= n_items) continue;
          touched.clear();
          for (int g : member[a]) touched.push_back(g);
          for (int g : member[b])
            if (std::find(touched.begin(), touched.end(), g) == touched.end()) touched.push_back(g);
          long before = 0, after = 0;
          for (int g : touched) before += cost[g];
          std::swap(colour[a], colour[b]);
          int fresh[64];
          for (size_t i = 0; i < touched.size(); ++i) {
            fresh[i] = group_cost(groups[touched[i]].data(), 8, colour);
            after += fresh[i];
          }
          if (after < before || (after == before && (rng.next() & 7) == 0)) {
            for (size_t i = 0; i < touched.size(); ++i) cost[touched[i]] = fresh[i];
          } else {
            std::swap(colour[a], colour[b]);
          }
        }
  }
};

}  // namespace sched_detail

// Proper 8-edge-colouring of a bipartite multigraph with maximum degree <= 8 (alternating-path
// recolouring).  edges[e] = (left node, right node); returns the colour of every edge.
inline std::vector<int> bipartite_edge_colouring8(int n_left, int n_right,
                                                  const std::vector<std::pair<int, int>> &edges) {
  std::vector<std::array<int, 8>> lcol(static_cast<size_t>(n_left)), rcol(static_cast<size_t>(n_right));
  for (auto &a : lcol) a.fill(-1);
  for (auto &a : rcol) a.fill(-1);
  std::vector<int> colour(edges.size(), -1);
  std::vector<int> path;
  for (size_t e = 0; e < edges.size(); ++e) {
    const int u = edges[e].first, w = edges[e].second;
    int a = -1, b = -1;
    for (int c = 0; c < 8 && a < 0; ++c)
      if (lcol[u][c] < 0) a = c;
    for (int c = 0; c < 8 && b < 0; ++c)
      if (rcol[w][c] < 0) b = c;
    if (a < 0 || b < 0) return {};   // degree above 8: caller checks
    if (rcol[w][a] >= 0) {
      // a is busy at w: swap a <-> b along the alternating path that starts at w with colour a
      path.clear();
      int node = w, want = a;
      bool at_right = true;
      while (true) {
        const int pe = at_right ? rcol[node][want] : lcol[node][want];
        if (pe < 0) break;
        path.push_back(pe);
        node = at_right ? edges[pe].first : edges[pe].second;
        at_right = !at_right;
        want = want == a ? b : a;
      }
      for (int pe : path) {
        lcol[edges[pe].first][colour[pe]] = -1;
        rcol[edges[pe].second][colour[pe]] = -1;
      }
      for (int pe : path) {
        colour[pe] = colour[pe] == a ? b : a;
        lcol[edges[pe].first][colour[pe]] = pe;
        rcol[edges[pe].second][colour[pe]] = pe;
      }
    }
    colour[e] = a;
    lcol[u][a] = int(e);
    rcol[w][a] = int(e);
  }
  return colour;
}

// Builds the schedule of one cell type.  X = rest positions [n][3].  Returns false (sched.valid
// stays false) when the type does not fit the scheduled kernel (the caller then uses another path).
inline bool build_local_schedule(const HostTypeData &h, const double *X, int tpt, LocalSchedule &out) {
  using namespace sched_detail;
  out = LocalSchedule();
  const int n = h.n, T = h.T;
  if (h.valence_max > 8 || tpt < 1 || tpt > 2) return false;
  const int ttri = ((T + tpt - 1) / tpt + 7) / 8 * 8;
  const int threads = (ttri + 31) / 32 * 32;      // triangle threads decide; a few vertices may take a 2nd pass
  // up to 32 overflow vertices: phase 0 in the last warp, phase C in the one before it
  if (n > threads + 32 || (n > threads && threads < 64)) return false;
  const int vstride = std::max(threads, (n + 31) / 32 * 32);
  const int maxv = h.valence_max <= 6 ? 6 : 8;
  const int n_vslots = (n + 7) / 8 * 8, n_tslots = tpt * ttri;
  const int octs_t = ttri / 8;                   // triangle octets per pass
  const int n_wgroups = tpt * 3 * octs_t;        // corner-force write groups (pass, corner, octet)
  const int n_cslots = 8 * n_wgroups + 8;        // + 8 zero slots, one per bank group
  if (threads > 1024 || n_vslots > 4096 || n_tslots > 4096 || n_cslots > 4096) return false;

  // scheduled triangle index tau = j*ttri + tid; identity map tau = t (tau >= T: idle)
  std::vector<int> rot(static_cast<size_t>(T), 0);
  auto corner = [&](int t, int c) { return h.tri[4 * t + (c + rot[t]) % 3]; };
  auto nbr = [&](int t, int s) { return h.tri_nbr[4 * t + (s + rot[t]) % 3]; };

  OctetColouring vc, tc;
  vc.init(n);
  tc.init(n_tslots);
  Lcg rng(uint64_t(n) * 1315423911u + uint64_t(T));
  auto build_groups = [&]() {
    std::vector<std::array<int, 8>> vg, ng;
    for (int k = 0; k < 3; ++k)
      for (int o = 0; o < n_tslots; o += 8) {
        std::array<int, 8> a, b;
        for (int i = 0; i < 8; ++i) {
          const int t = o + i;
          a[i] = t < T ? corner(t, k) : -1;
          b[i] = t < T ? nbr(t, k) : -1;
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
    for (int s = 0; s < sweeps; ++s) {
      vc.sweep(rng);
      tc.sweep(rng);
    }
    // best cyclic rotation of the 8 triangles of every octet, colours fixed (3^8 combinations)
    for (int o = 0; o < n_tslots; o += 8) {
      const int cnt = std::min(8, T - o);
      if (cnt <= 0) continue;
      int best_cost = 1 << 30, best_combo = 0, n_combo = 1;
      for (int i = 0; i < cnt; ++i) n_combo *= 3;
      for (int combo = 0; combo < n_combo; ++combo) {
        int cc = combo, cost = 0, rr[8];
        for (int i = 0; i < cnt; ++i) { rr[i] = cc % 3; cc /= 3; }
        for (int k = 0; k < 3 && cost < best_cost; ++k) {
          int vi[8], ti[8];
          for (int i = 0; i < cnt; ++i) {
            vi[i] = h.tri[4 * (o + i) + (k + rr[i]) % 3];
            ti[i] = h.tri_nbr[4 * (o + i) + (k + rr[i]) % 3];
          }
          cost += group_cost(vi, cnt, vc.colour) + group_cost(ti, cnt, tc.colour);
        }
        if (cost < best_cost) { best_cost = cost; best_combo = combo; }
      }
      for (int i = 0; i < cnt; ++i) { rot[o + i] = best_combo % 3; best_combo /= 3; }
    }
  }
  build_groups();
  for (int s = 0; s < sweeps; ++s) {
    vc.sweep(rng);
    tc.sweep(rng);
  }
  out.wf_vertex = 4.0 * double(vc.total()) / double(vc.groups.size());
  out.wf_normal = 4.0 * double(tc.total()) / double(tc.groups.size());
  auto vslot = [&](int v) { return 8 * (v / 8) + vc.colour[v]; };
  auto tslot = [&](int t) { return 8 * (t / 8) + tc.colour[t]; };

  // ---- corner-force slots: exact bipartite edge colouring ----------------------------------
  std::vector<int> fill(static_cast<size_t>(n), 0);
  std::vector<int> read_pos(size_t(T) * 3);                 // k = position in the vertex's read list
  std::vector<std::pair<int, int>> edges(size_t(T) * 3);
  const int octs_v = n_vslots / 8;
  for (int t = 0; t < T; ++t)
    for (int c = 0; c < 3; ++c) {
      const int v = corner(t, c), k = fill[v]++;
      read_pos[3 * t + c] = k;
      const int j = t / ttri, oct = (t % ttri) / 8;
      edges[3 * t + c] = {(j * 3 + c) * octs_t + oct, k * octs_v + v / 8};
    }
  const std::vector<int> ecol = bipartite_edge_colouring8(n_wgroups, maxv * octs_v, edges);
  if (ecol.size() != edges.size()) return false;
  auto cslot = [&](int t, int c) { return 8 * edges[3 * t + c].first + ecol[3 * t + c]; };

  // ---- tables --------------------------------------------------------------------------------
  out.threads = threads; out.vstride = vstride; out.tpt = tpt; out.ttri = ttri; out.maxv = maxv;
  out.n_vslots = n_vslots; out.n_tslots = n_tslots; out.n_cslots = n_cslots;
  out.tri_words.assign(size_t(tpt) * 5 * threads, 0u);
  out.tri_consts.assign(size_t(tpt) * 12 * threads, 0.f);
  const int vwords = 1 + maxv / 2;
  out.vtx_words.assign(size_t(vwords) * vstride, 0u);
  out.vtx_coef.assign(size_t(vstride), 0.f);
  const npfem_material &m = h.mat;
  const double B4 = m.skalak_B / 4.0, C4 = m.skalak_C / 4.0;
  for (int t = 0; t < T; ++t) {
    const int j = t / ttri, tid = t % ttri;
    auto W = [&](int q) -> uint32_t & { return out.tri_words[(size_t(j) * 5 + q) * threads + tid]; };
    auto K = [&](int q) -> float & { return out.tri_consts[(size_t(j) * 12 + q) * threads + tid]; };
    const uint32_t v0 = 16u * vslot(corner(t, 0)), v1 = 16u * vslot(corner(t, 1)), v2 = 16u * vslot(corner(t, 2));
    const uint32_t n0 = 16u * tslot(nbr(t, 0)), n1 = 16u * tslot(nbr(t, 1)), n2 = 16u * tslot(nbr(t, 2));
    const uint32_t c0 = 16u * cslot(t, 0), c1 = 16u * cslot(t, 1), c2 = 16u * cslot(t, 2);
    W(0) = v0 | (v1 << 16);
    W(1) = v2 | (n0 << 16);
    W(2) = n1 | (n2 << 16);
    W(3) = c0 | (c1 << 16);
    W(4) = c2 | ((16u * tslot(t)) << 16);
    // rest data of the ROTATED triangle: Dm^-1 = [[a, b], [0, c]] (reading R5), A0
    const double *x0 = X + 3 * corner(t, 0), *x1 = X + 3 * corner(t, 1), *x2 = X + 3 * corner(t, 2);
    double E1[3], E2[3], N[3];
    for (int q = 0; q < 3; ++q) { E1[q] = x1[q] - x0[q]; E2[q] = x2[q] - x0[q]; }
    cross3(E1, E2, N);
    const double len1 = std::sqrt(dot3(E1, E1)), twoA = std::sqrt(dot3(N, N));
    const double a = 1.0 / len1, height = twoA / len1, c = 1.0 / height;
    const double b = -(dot3(E2, E1) / len1) / (len1 * height), A0 = 0.5 * twoA;
    const double J = (a * c) * (a * c);
    K(0) = float(a * a + b * b);            // R11   (R = Dm^-1 Dm^-T)
    K(1) = float(b * c);                    // R12
    K(2) = float(c * c);                    // R22
    K(3) = float(J);                        // det(Dm^-1)^2
    K(4) = float(2.0 * A0 * B4);            // tA
    K(5) = float(2.0 * A0 * J * C4);        // tC
    for (int s = 0; s < 3; ++s) {
      const int so = (s + rot[t]) % 3;      // the hinge angle belongs to the edge, not to the rotation
      K(6 + s) = float(m.k_bending * h.hinge_rest[6 * t + 2 * so + 0]);
      K(9 + s) = float(m.k_bending * h.hinge_rest[6 * t + 2 * so + 1]);
    }
  }
  {   // bound of a thread's partial of 6V = sum_t x_0 . (e_1 x e_2) in cell-local (centroid) coordinates
    double cen[3] = {0, 0, 0}, rmax = 0, bound = 0;
    for (int v = 0; v < n; ++v)
      for (int q = 0; q < 3; ++q) cen[q] += X[3 * v + q] / n;
    for (int v = 0; v < n; ++v) {
      double r2 = 0;
      for (int q = 0; q < 3; ++q) r2 += (X[3 * v + q] - cen[q]) * (X[3 * v + q] - cen[q]);
      rmax = std::max(rmax, std::sqrt(r2));
    }
    for (int tid = 0; tid < ttri; ++tid) {
      double sum = 0;
      for (int j = 0; j < tpt; ++j)
        if (j * ttri + tid < T) sum += rmax * 2.0 * h.tri_rest[4 * (j * ttri + tid) + 3];
      bound = std::max(bound, sum);
    }
    out.vol_lane_bound = bound;
  }
  // vertex reads: real corner slots, then zero slots of a bank group the read group does not use
  std::vector<std::array<int, 8>> reads(static_cast<size_t>(n));
  for (auto &r : reads) r.fill(-1);
  for (int t = 0; t < T; ++t)
    for (int c = 0; c < 3; ++c) reads[corner(t, c)][read_pos[3 * t + c]] = cslot(t, c);
  for (int k = 0; k < maxv; ++k)
    for (int o = 0; o < n; o += 8) {
      bool used[8] = {false, false, false, false, false, false, false, false};
      for (int v = o; v < std::min(o + 8, n); ++v)
        if (reads[v][k] >= 0) used[reads[v][k] % 8] = true;
      int free_colour = 0;
      while (free_colour < 7 && used[free_colour]) ++free_colour;
      for (int v = o; v < std::min(o + 8, n); ++v)
        if (reads[v][k] < 0) reads[v][k] = 8 * n_wgroups + free_colour;
    }
  const double gamma = (m.rayleigh_beta / h.h) / (1.0 + m.rayleigh_beta / h.h);
  const double inertia = (1.0 + h.h * m.rayleigh_alpha) / (h.h * h.h);
  for (int v = 0; v < n; ++v) {
    out.vtx_words[v] = 16u * uint32_t(vslot(v));
    for (int q = 0; q < maxv / 2; ++q)
      out.vtx_words[size_t(1 + q) * vstride + v] =
          (16u * uint32_t(reads[v][2 * q])) | ((16u * uint32_t(reads[v][2 * q + 1])) << 16);
    out.vtx_coef[v] = float((1.0 - gamma) * inertia * h.mass[v]);
  }
  out.valid = true;
  return true;
}

}  // namespace npfem
