// Create-time schedule of the fp32 "quad" local step (local_quad.cu): one thread per PAIR of adjacent triangles.
//
// Why (profiles/r2_ncu.md): the scheduled kernel's triangle phases are issue-bound and its vertex phases are bound by
// shared-memory wavefronts; what is left is less work per cell.  A thread that owns two triangles sharing an edge
//   T0 = (p, q, r),  T1 = (p, s, q)          (shared edge p-q, both counter-clockwise)
// gathers 4 vertex positions and 4 neighbour normals instead of 6 + 6, evaluates the shared hinge once, and stores 4
// corner forces instead of 6 (the two triangles' forces on p and on q are summed in registers), so a vertex gathers one
// slot per incident QUAD (4 on average) instead of one per incident triangle (6).  A perfect matching of the dual graph
// exists for every closed triangulated surface (it is cubic and bridgeless: Petersen); it is found by Edmonds'
// blossom algorithm, then improved by alternating-cycle flips that lower the largest number of quads at a vertex.
// Slot assignment (conflict-free gathers and stores) is the machinery of local_schedule.hpp over quads.
// Everything here is integer / fp64 host work done once per cell TYPE.  Product code: shares nothing with oracle/.
#pragma once

#include <algorithm>
#include <array>
#include <cmath>
#include <cstdint>
#include <vector>

#include "host_setup.hpp"
#include "local_schedule.hpp"

namespace npfem {

struct QuadSchedule {
  bool valid = false;
  int threads = 0;    // CTA size (multiple of 32); quad q and vertex q are owned by thread q
  int vstride = 0;    // row stride of the vertex tables (>= n)
  int nq = 0;         // quads = T / 2
  int qthreads = 0;   // threads that own a quad slot (multiple of 8, >= nq)
  int maxq = 0;       // corner-force reads per vertex (6 or 8)
  int n_vslots = 0, n_tslots = 0, n_cslots = 0;   // float4 slots of sx / sN / sC
  std::vector<uint32_t> quad_words;   // [7][threads] packed 16-bit byte offsets (see local_quad.cu)
  std::vector<float> quad_consts;     // [22][threads]
  std::vector<uint32_t> vtx_words;    // [1 + maxq/2][vstride] own slot, corner-force slots
  std::vector<float> vtx_coef;        // [vstride]
  std::vector<int> mate;              // [T] the matching (for the consistency check)
  double wf_vertex = 0, wf_normal = 0;   // predicted wavefronts per gather instruction (ideal 4)
  double vol_lane_bound = 0;
  int quads_at_vertex_max = 0;
  double quads_at_vertex_mean = 0;
};

namespace quad_detail {

// Maximum matching in a general graph (Edmonds' blossom algorithm, BFS version, O(V^3) worst case; the dual
// graph of a mesh has 3 neighbours per node and starts from a greedy matching, so it is fast in practice).
struct Blossom {
  int n;
  const std::vector<std::array<int, 3>> &adj;
  std::vector<int> match, parent, base, queue;
  std::vector<char> used, blossom;
  Blossom(int n_, const std::vector<std::array<int, 3>> &a) : n(n_), adj(a), match(size_t(n_), -1), parent(size_t(n_)),
                                                               base(size_t(n_)), used(size_t(n_)), blossom(size_t(n_)) {}
  int lca(int a, int b) {
    std::vector<char> seen(size_t(n), 0);
    for (;;) {
      a = base[a];
      seen[a] = 1;
      if (match[a] < 0) break;
      a = parent[match[a]];
    }
    for (;;) {
      b = base[b];
      if (seen[b]) return b;
      b = parent[match[b]];
    }
  }
  void mark_path(int v, int b, int child) {
    while (base[v] != b) {
      blossom[base[v]] = blossom[base[match[v]]] = 1;
      parent[v] = child;
      child = match[v];
      v = parent[match[v]];
    }
  }
  int find_path(int root) {
    std::fill(used.begin(), used.end(), 0);
    std::fill(parent.begin(), parent.end(), -1);
    for (int i = 0; i < n; ++i) base[i] = i;
    queue.clear();
    queue.push_back(root);
    used[root] = 1;
    for (size_t qh = 0; qh < queue.size(); ++qh) {
      const int v = queue[qh];
      for (int to : adj[v]) {
        if (to < 0 || base[v] == base[to] || match[v] == to) continue;
        if (to == root || (match[to] >= 0 && parent[match[to]] >= 0)) {
          const int cur = lca(v, to);
          std::fill(blossom.begin(), blossom.end(), 0);
          mark_path(v, cur, to);
          mark_path(to, cur, v);
          for (int i = 0; i < n; ++i)
            if (blossom[base[i]]) {
              base[i] = cur;
              if (!used[i]) {
                used[i] = 1;
                queue.push_back(i);
              }
            }
        } else if (parent[to] < 0) {
          parent[to] = v;
          if (match[to] < 0) return to;
          used[match[to]] = 1;
          queue.push_back(match[to]);
        }
      }
    }
    return -1;
  }
  // returns the number of matched pairs; `match` may hold a partial matching to start from
  int solve() {
    for (int v = 0; v < n; ++v)      // greedy completion
      if (match[v] < 0)
        for (int to : adj[v])
          if (to >= 0 && match[to] < 0) {
            match[v] = to;
            match[to] = v;
            break;
          }
    for (int v = 0; v < n; ++v)
      if (match[v] < 0) {
        int u = find_path(v);
        while (u >= 0) {
          const int pv = parent[u], ppv = match[pv];
          match[u] = pv;
          match[pv] = u;
          u = ppv;
        }
      }
    int pairs = 0;
    for (int v = 0; v < n; ++v) pairs += match[v] >= 0;
    return pairs / 2;
  }
};

// A partial matching that gives every vertex matched edges: pass k = 1, 2 visits the vertices in order and, if a vertex
// has fewer than k matched incident edges, pairs two still unmatched adjacent triangles of its fan.  With two matched
// edges at every vertex (the regular-lattice pattern: rhombi along one direction) a valence-6 vertex sees 4 quads.
inline void seed_matching(const HostTypeData &h, std::vector<int> &mate) {
  mate.assign(size_t(h.T), -1);
  std::vector<std::vector<int>> fan(size_t(h.n));
  for (int t = 0; t < h.T; ++t)
    for (int c = 0; c < 3; ++c) fan[h.tri[4 * t + c]].push_back(t);
  std::vector<int> matched_at(size_t(h.n), 0);
  for (int pass = 1; pass <= 2; ++pass)
    for (int v = 0; v < h.n; ++v) {
      if (matched_at[v] >= pass) continue;
      bool done = false;
      for (size_t i = 0; i < fan[v].size() && !done; ++i) {
        const int a = fan[v][i];
        if (mate[a] >= 0) continue;
        for (int s = 0; s < 3 && !done; ++s) {
          const int b = h.tri_nbr[4 * a + s];
          const int u0 = h.tri[4 * a + s], u1 = h.tri[4 * a + (s + 1) % 3];     // the shared edge
          if (b < 0 || mate[b] >= 0 || (u0 != v && u1 != v)) continue;
          const int w = u0 == v ? u1 : u0;
          if (matched_at[w] >= 2) continue;                                     // do not overload the other endpoint
          mate[a] = b;
          mate[b] = a;
          ++matched_at[v];
          ++matched_at[w];
          done = true;
        }
      }
    }
}

// For a matching `mate`, the number of quads incident to every vertex: valence - (matched edges at the vertex).
inline std::vector<int> quads_at_vertices(const HostTypeData &h, const std::vector<int> &mate) {
  std::vector<int> cnt(size_t(h.n), 0);
  for (int t = 0; t < h.T; ++t)
    for (int c = 0; c < 3; ++c) ++cnt[h.tri[4 * t + c]];                 // valence = incident triangles
  for (int t = 0; t < h.T; ++t)
    if (mate[t] > t)
      for (int s = 0; s < 3; ++s)
        if (h.tri_nbr[4 * t + s] == mate[t]) {                           // the shared edge v_s - v_{s+1}
          --cnt[h.tri[4 * t + s]];
          --cnt[h.tri[4 * t + (s + 1) % 3]];
          break;
        }
  return cnt;
}

// Alternating-cycle flips around primal vertices: the triangles around a vertex form a cycle in the dual graph; if the
// fan contains matched pairs (t_i, t_{i+1}) and the fan has even length with EVERY second edge matched, rotating the
// matching along the fan keeps the count at that vertex but moves the matched primal edges to other neighbours.  More
// generally any alternating 4-cycle A-B (matched), B-C, C-D (matched), D-A can be flipped to B-C, D-A.  The search flips
// a 4-cycle whenever it lowers  sum_v max(0, quads(v) - 4)^2  (quads(v) = 4 is the regular-lattice value).
inline void improve_matching(const HostTypeData &h, std::vector<int> &mate, int sweeps) {
  auto shared_edge = [&](int a, int b, int &u, int &v) {
    for (int s = 0; s < 3; ++s)
      if (h.tri_nbr[4 * a + s] == b) {
        u = h.tri[4 * a + s];
        v = h.tri[4 * a + (s + 1) % 3];
        return true;
      }
    return false;
  };
  std::vector<int> cnt = quads_at_vertices(h, mate);
  auto pen = [](int c) { return c > 4 ? (c - 4) * (c - 4) : 0; };
  for (int sweep = 0; sweep < sweeps; ++sweep) {
    bool any = false;
    for (int a = 0; a < h.T; ++a) {
      const int b = mate[a];
      if (b < 0) continue;
      for (int sb = 0; sb < 3; ++sb) {
        const int c = h.tri_nbr[4 * b + sb];
        if (c == a || c < 0) continue;
        const int d = mate[c];
        if (d < 0 || d == a || d == b) continue;
        bool closes = false;                                             // D adjacent to A?
        for (int s = 0; s < 3; ++s) closes |= h.tri_nbr[4 * d + s] == a;
        if (!closes) continue;
        int e[4][2];
        if (!shared_edge(a, b, e[0][0], e[0][1]) || !shared_edge(c, d, e[1][0], e[1][1]) ||
            !shared_edge(b, c, e[2][0], e[2][1]) || !shared_edge(d, a, e[3][0], e[3][1]))
          continue;
        // flip: edges 0, 1 leave the matching (their endpoints gain a quad), edges 2, 3 enter it
        int touched[8], delta[8], nt = 0;
        auto add = [&](int v, int dl) {
          for (int i = 0; i < nt; ++i)
            if (touched[i] == v) { delta[i] += dl; return; }
          touched[nt] = v; delta[nt] = dl; ++nt;
        };
        for (int k = 0; k < 2; ++k) { add(e[k][0], +1); add(e[k][1], +1); }
        for (int k = 2; k < 4; ++k) { add(e[k][0], -1); add(e[k][1], -1); }
        int before = 0, after = 0;
        for (int i = 0; i < nt; ++i) { before += pen(cnt[touched[i]]); after += pen(cnt[touched[i]] + delta[i]); }
        if (after < before) {
          mate[b] = c; mate[c] = b; mate[d] = a; mate[a] = d;
          for (int i = 0; i < nt; ++i) cnt[touched[i]] += delta[i];
          any = true;
          break;                                                         // a's mate changed: next triangle
        }
      }
    }
    if (!any) break;
  }
}

// Repair of the vertices that see the most quads (a valence-6 vertex none of whose edges is matched sees 6): pair two
// adjacent triangles of its fan by force, which frees their two old mates, and reconnect those by an augmenting path
// (Edmonds again, from the one free triangle to the other).  A move is kept if it lowers the lexicographic cost
// (vertices at the maximum, sum of squared excess over 4).  Deterministic: vertices and fan pairs in index order.
inline void repair_matching(const HostTypeData &h, const std::vector<std::array<int, 3>> &adj, std::vector<int> &mate,
                            int rounds) {
  auto cost = [&](const std::vector<int> &m, int &worst, long &n_worst, long &excess) {
    const std::vector<int> cnt = quads_at_vertices(h, m);
    worst = 0;
    for (int c : cnt) worst = std::max(worst, c);
    n_worst = excess = 0;
    for (int c : cnt) {
      n_worst += c == worst;
      excess += c > 4 ? long(c - 4) * (c - 4) : 0;
    }
  };
  sched_detail::Lcg rng(uint64_t(h.n) * 2654435761u + uint64_t(h.T));
  std::vector<int> best = mate, sideways;
  int best_w, n_sideways = 0;
  long best_n, best_e;
  cost(mate, best_w, best_n, best_e);
  for (int round = 0; round < rounds; ++round) {
    int worst;
    long n_worst, excess;
    cost(mate, worst, n_worst, excess);
    if (worst <= 4) break;
    const std::vector<int> cnt = quads_at_vertices(h, mate);
    bool improved = false;
    sideways.clear();
    for (int v = 0; v < h.n && !improved; ++v) {
      if (cnt[v] != worst) continue;
      for (int a = 0; a < h.T && !improved; ++a) {                      // fan of v: triangles that contain v
        bool has = false;
        for (int c = 0; c < 3; ++c) has |= h.tri[4 * a + c] == v;
        if (!has) continue;
        for (int s = 0; s < 3 && !improved; ++s) {
          const int b = h.tri_nbr[4 * a + s];
          const int u0 = h.tri[4 * a + s], u1 = h.tri[4 * a + (s + 1) % 3];
          if (b < a || mate[a] == b || (u0 != v && u1 != v)) continue;    // the shared edge must end at v
          Blossom bl(h.T, adj);
          bl.match = mate;
          const int ma = mate[a], mb = mate[b];
          bl.match[a] = b; bl.match[b] = a; bl.match[ma] = -1; bl.match[mb] = -1;
          int u = bl.find_path(ma);
          if (u < 0) continue;
          while (u >= 0) {
            const int pv = bl.parent[u], ppv = bl.match[pv];
            bl.match[u] = pv;
            bl.match[pv] = u;
            u = ppv;
          }
          int w2;
          long n2, e2;
          cost(bl.match, w2, n2, e2);
          if (w2 < worst || (w2 == worst && (n2 < n_worst || (n2 == n_worst && e2 < excess)))) {
            mate = bl.match;
            improved = true;
          } else if (w2 == worst && n2 == n_worst && (rng.next() % 3) == 0) {
            sideways = bl.match;                                          // a move that does not hurt: kept in reserve
          }
        }
      }
    }
    if (!improved) {
      if (sideways.empty() || ++n_sideways > rounds / 4) break;           // plateau: step sideways a few times
      mate = sideways;
    }
    int w;
    long nw, ex;
    cost(mate, w, nw, ex);
    if (w < best_w || (w == best_w && (nw < best_n || (nw == best_n && ex < best_e)))) {
      best = mate; best_w = w; best_n = nw; best_e = ex;
    }
  }
  mate = best;
}

}  // namespace quad_detail

// Builds the quad schedule of one cell type.  X = rest positions [n][3].  Returns false (valid stays false) when the
// type does not fit the quad kernel (odd triangle count, no perfect matching, too large: the caller uses another path).
inline bool build_quad_schedule(const HostTypeData &h, const double *X, QuadSchedule &out) {
  using namespace sched_detail;
  using namespace quad_detail;
  out = QuadSchedule();
  const int n = h.n, T = h.T;
  if (h.valence_max > 8 || (T & 1)) return false;
  const int nq = T / 2;
  const int qthreads = (nq + 7) / 8 * 8;
  const int threads = (qthreads + 31) / 32 * 32;
  if (threads > 1024 || n > threads + 32 || (n > threads && threads < 64)) return false;
  const int vstride = std::max(threads, (n + 31) / 32 * 32);
  const int n_vslots = (n + 7) / 8 * 8, n_tslots = 2 * qthreads;
  const int octs_q = qthreads / 8;
  const int n_wgroups = 4 * octs_q;                 // corner-force write groups (role, octet)
  const int n_cslots = 8 * n_wgroups + 8;           // + 8 zero slots, one per bank group
  if (n_vslots > 4096 || n_tslots > 4096 || n_cslots > 4096) return false;

  // ---- matching ------------------------------------------------------------------------------
  std::vector<std::array<int, 3>> adj(static_cast<size_t>(T));
  for (int t = 0; t < T; ++t) adj[t] = {h.tri_nbr[4 * t], h.tri_nbr[4 * t + 1], h.tri_nbr[4 * t + 2]};
  Blossom bl(T, adj);
  if (bl.solve() != nq) return false;
  std::vector<int> mate = bl.match;
  repair_matching(h, adj, mate, 120);
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

  // ---- corner-force slots: exact bipartite edge colouring ({write groups} x {read groups}, degree <= 8) ----------
  std::vector<int> fill(static_cast<size_t>(n), 0);
  std::vector<int> read_pos(size_t(nq) * 4);
  std::vector<std::pair<int, int>> edges(size_t(nq) * 4);
  const int octs_v = n_vslots / 8;
  for (int k = 0; k < nq; ++k) {
    const Roles R = roles(k);
    const int vs[4] = {R.p, R.q, R.r, R.s};
    for (int role = 0; role < 4; ++role) {
      const int v = vs[role], pos = fill[v]++;
      if (pos >= maxq) return false;
      read_pos[4 * k + role] = pos;
      edges[4 * k + role] = {role * octs_q + k / 8, pos * octs_v + v / 8};
    }
  }
  const std::vector<int> ecol = bipartite_edge_colouring8(n_wgroups, maxq * octs_v, edges);
  if (ecol.size() != edges.size()) return false;
  auto cslot = [&](int k, int role) { return 8 * edges[4 * k + role].first + ecol[4 * k + role]; };

  // ---- tables --------------------------------------------------------------------------------
  out.threads = threads; out.vstride = vstride; out.nq = nq; out.qthreads = qthreads; out.maxq = maxq;
  out.n_vslots = n_vslots; out.n_tslots = n_tslots; out.n_cslots = n_cslots;
  out.quad_words.assign(size_t(7) * threads, 0u);
  out.quad_consts.assign(size_t(22) * threads, 0.f);
  const int vwords = 1 + maxq / 2;
  out.vtx_words.assign(size_t(vwords) * vstride, 0u);
  out.vtx_coef.assign(size_t(vstride), 0.f);
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
  for (int k = 0; k < nq; ++k) {
    const Roles R = roles(k);
    auto W = [&](int q) -> uint32_t & { return out.quad_words[size_t(q) * threads + k]; };
    auto K = [&](int q) -> float & { return out.quad_consts[size_t(q) * threads + k]; };
    W(0) = 16u * vslot(R.p) | (16u * vslot(R.q)) << 16;
    W(1) = 16u * vslot(R.r) | (16u * vslot(R.s)) << 16;
    W(2) = 16u * tslot(R.n0) | (16u * tslot(R.n1)) << 16;
    W(3) = 16u * tslot(R.n2) | (16u * tslot(R.n3)) << 16;
    W(4) = 16u * tslot(R.A) | (16u * tslot(R.B)) << 16;
    W(5) = 16u * cslot(k, 0) | (16u * cslot(k, 1)) << 16;
    W(6) = 16u * cslot(k, 2) | (16u * cslot(k, 3)) << 16;
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
    out.vol_lane_bound = std::max(out.vol_lane_bound, rmax * 2.0 * (A0 + A1));
  }
  // vertex reads: real corner slots, then zero slots of a bank group the read group does not use
  std::vector<std::array<int, 8>> reads(static_cast<size_t>(n));
  for (auto &r : reads) r.fill(-1);
  for (int k = 0; k < nq; ++k) {
    const Roles R = roles(k);
    const int vs[4] = {R.p, R.q, R.r, R.s};
    for (int role = 0; role < 4; ++role) reads[vs[role]][read_pos[4 * k + role]] = cslot(k, role);
  }
  for (int k = 0; k < maxq; ++k)
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
    for (int q = 0; q < maxq / 2; ++q)
      out.vtx_words[size_t(1 + q) * vstride + v] =
          (16u * uint32_t(reads[v][2 * q])) | ((16u * uint32_t(reads[v][2 * q + 1])) << 16);
    out.vtx_coef[v] = float((1.0 - gamma) * inertia * h.mass[v]);
  }
  out.valid = true;
  return true;
}

}  // namespace npfem
