// Host-side (fp64) per-cell-TYPE precompute for npfem_create: topology tables, rest data,
// one-ring cotangent operator, lumped mass and the dense constant matrix H~.
//
// Follows PAPER.md:257-272 (Eqs. 1-4) with the readings R4-R11 of DESIGN.md:
//   Dm^-1 = [[a,b],[0,c]] and A0 per triangle; hinge rest angles; V0, A, A_v;
//   L_cot = sum_t A0 G_t G_t^T;  L = (B+2C) L_cot + k_b L_cot diag(1/A_v) L_cot;
//   M = diag(rho V0 A_v / A);  M~ = (1+h alpha) M + h beta L;  H~ = M~/h^2 + L.
// Product code: shares nothing with oracle/.
#pragma once

#include <cmath>
#include <cstdint>
#include <string>
#include <unordered_map>
#include <vector>

#include "../../include/npfem.h"

namespace npfem {

struct HostTypeData {
  int n = 0, T = 0, n_pad = 0, valence_max = 0;
  npfem_material mat{};
  double h = 0;
  double V0 = 0, A = 0;
  std::vector<int32_t> tri;         // [T][4]  v0, v1, v2, 0
  std::vector<int32_t> tri_nbr;     // [T][4]  triangle across edge s (v_s -> v_{s+1}), s = 0..2, 0
  std::vector<double> tri_rest;     // [T][4]  a, b, c, A0
  std::vector<double> hinge_rest;   // [T][6]  (cos theta0, sin theta0) for edge s = 0..2
  std::vector<int32_t> vtx_corner;  // [valence_max][n] corner id 3t+c incident to vertex, -1 = none
  std::vector<int32_t> vtx_nbr;     // [valence_max][n] one-ring neighbour, own index if none
  std::vector<double> vtx_w;        // [valence_max+1][n] L_cot row: [0] diagonal, [1+q] neighbour q
  std::vector<double> area_v;       // [n]
  std::vector<double> mass;         // [n]
  std::vector<double> H;            // [n][n] dense H~
};

inline void cross3(const double *u, const double *v, double *w) {
  w[0] = u[1] * v[2] - u[2] * v[1];
  w[1] = u[2] * v[0] - u[0] * v[2];
  w[2] = u[0] * v[1] - u[1] * v[0];
}
inline double dot3(const double *u, const double *v) { return u[0] * v[0] + u[1] * v[1] + u[2] * v[2]; }

// Returns NPFEM_OK or NPFEM_EMESH/NPFEM_EINVAL with `err` filled.
inline int build_host_type(const npfem_cell_type &ct, double h, HostTypeData &out, std::string &err) {
  const int n = ct.n_vertices, T = ct.n_triangles;
  if (n < 4 || T < 4 || !ct.rest_positions || !ct.triangles) {
    err = "cell type needs >= 4 vertices, >= 4 triangles and non-null arrays";
    return NPFEM_EINVAL;
  }
  if (n > 65535 || T > 65535 * 2) {
    err = "cell type too large (n_vertices must be <= 65535)";
    return NPFEM_EINVAL;
  }
  const npfem_material &m = ct.material;
  if (!(m.density > 0) || !(h > 0) || m.skalak_B < 0 || m.skalak_C < 0 || m.k_bending < 0 ||
      m.k_volume < 0 || m.rayleigh_alpha < 0 || m.rayleigh_beta < 0 || m.kappa_damping < 0 ||
      m.kappa_damping > 1) {
    err = "material constants must be non-negative, density and dt positive, kappa in [0,1]";
    return NPFEM_EINVAL;
  }
  out.n = n;
  out.T = T;
  out.n_pad = (n + 15) / 16 * 16;
  out.mat = m;
  out.h = h;
  const double *X = ct.rest_positions;

  // ---- half-edge map: directed edge (u,v) -> 3*t + s ------------------------------------
  std::unordered_map<uint64_t, int32_t> half;
  half.reserve(size_t(T) * 3 * 2);
  out.tri.assign(size_t(T) * 4, 0);
  std::vector<int> valence(n, 0);
  for (int t = 0; t < T; ++t) {
    int v[3];
    for (int c = 0; c < 3; ++c) {
      v[c] = ct.triangles[3 * t + c];
      if (v[c] < 0 || v[c] >= n) {
        err = "triangle " + std::to_string(t) + " references vertex out of range";
        return NPFEM_EMESH;
      }
      out.tri[4 * t + c] = v[c];
    }
    if (v[0] == v[1] || v[1] == v[2] || v[0] == v[2]) {
      err = "triangle " + std::to_string(t) + " is degenerate (repeated vertex)";
      return NPFEM_EMESH;
    }
    for (int s = 0; s < 3; ++s) {
      uint64_t key = (uint64_t(uint32_t(v[s])) << 32) | uint32_t(v[(s + 1) % 3]);
      if (!half.emplace(key, 3 * t + s).second) {
        err = "directed edge appears twice: surface is not consistently oriented / not manifold";
        return NPFEM_EMESH;
      }
      valence[v[s]]++;
    }
  }
  out.tri_nbr.assign(size_t(T) * 4, 0);
  for (int t = 0; t < T; ++t)
    for (int s = 0; s < 3; ++s) {
      uint64_t twin = (uint64_t(uint32_t(out.tri[4 * t + (s + 1) % 3])) << 32) | uint32_t(out.tri[4 * t + s]);
      auto it = half.find(twin);
      if (it == half.end()) {
        err = "edge without a twin: surface is not closed";
        return NPFEM_EMESH;
      }
      out.tri_nbr[4 * t + s] = it->second / 3;
    }
  int vmax = 0;
  for (int v = 0; v < n; ++v) {
    if (valence[v] < 3) {
      err = "vertex " + std::to_string(v) + " has fewer than 3 incident triangles";
      return NPFEM_EMESH;
    }
    vmax = valence[v] > vmax ? valence[v] : vmax;
  }
  if (vmax > 32) {
    err = "vertex valence above 32 is not supported";
    return NPFEM_EMESH;
  }
  out.valence_max = vmax;

  // ---- rest data per triangle ------------------------------------------------------------
  out.tri_rest.assign(size_t(T) * 4, 0.0);
  out.area_v.assign(n, 0.0);
  std::vector<double> normal(size_t(T) * 3);
  double V0 = 0, A = 0;
  for (int t = 0; t < T; ++t) {
    const double *x0 = X + 3 * out.tri[4 * t], *x1 = X + 3 * out.tri[4 * t + 1], *x2 = X + 3 * out.tri[4 * t + 2];
    double E1[3], E2[3], N[3];
    for (int c = 0; c < 3; ++c) {
      E1[c] = x1[c] - x0[c];
      E2[c] = x2[c] - x0[c];
    }
    cross3(E1, E2, N);
    const double len1 = std::sqrt(dot3(E1, E1));
    const double twoA = std::sqrt(dot3(N, N));
    if (!(len1 > 0) || !(twoA > 1e-14 * len1 * len1)) {
      err = "triangle " + std::to_string(t) + " has zero rest area";
      return NPFEM_EMESH;
    }
    const double proj = dot3(E2, E1) / len1;
    const double height = twoA / len1;
    out.tri_rest[4 * t + 0] = 1.0 / len1;                // a
    out.tri_rest[4 * t + 1] = -proj / (len1 * height);   // b
    out.tri_rest[4 * t + 2] = 1.0 / height;              // c
    out.tri_rest[4 * t + 3] = 0.5 * twoA;                // A0
    for (int c = 0; c < 3; ++c) {
      normal[3 * t + c] = N[c];
      out.area_v[out.tri[4 * t + c]] += 0.5 * twoA / 3.0;
    }
    A += 0.5 * twoA;
    V0 += dot3(x0, N) / 6.0;   // x0.(x1 x x2) = x0.((x1-x0) x (x2-x0))
  }
  if (!(V0 > 0)) {
    err = "enclosed rest volume is not positive: triangles must be counter-clockwise seen from outside";
    return NPFEM_EMESH;
  }
  out.V0 = V0;
  out.A = A;

  // ---- rest hinge angles, seen from each triangle's own edge -----------------------------
  out.hinge_rest.assign(size_t(T) * 6, 0.0);
  for (int t = 0; t < T; ++t)
    for (int s = 0; s < 3; ++s) {
      const int tb = out.tri_nbr[4 * t + s];
      const double *xi = X + 3 * out.tri[4 * t + s], *xj = X + 3 * out.tri[4 * t + (s + 1) % 3];
      double e[3] = {xj[0] - xi[0], xj[1] - xi[1], xj[2] - xi[2]};
      const double *NA = &normal[3 * t], *NB = &normal[3 * tb];
      double cr[3];
      cross3(NA, NB, cr);
      const double inv = 1.0 / std::sqrt(dot3(NA, NA) * dot3(NB, NB));
      out.hinge_rest[6 * t + 2 * s + 0] = dot3(NA, NB) * inv;
      out.hinge_rest[6 * t + 2 * s + 1] = dot3(cr, e) / std::sqrt(dot3(e, e)) * inv;
    }

  // ---- vertex incidence (corners) and one-ring neighbour lists ---------------------------
  out.vtx_corner.assign(size_t(vmax) * n, -1);
  out.vtx_nbr.assign(size_t(vmax) * n, 0);
  for (int q = 0; q < vmax; ++q)
    for (int v = 0; v < n; ++v) out.vtx_nbr[size_t(q) * n + v] = v;
  std::vector<int> fill_c(n, 0), fill_n(n, 0);
  auto nbr_slot = [&](int v, int u) -> int {   // slot of neighbour u in the list of v (append if new)
    for (int q = 0; q < fill_n[v]; ++q)
      if (out.vtx_nbr[size_t(q) * n + v] == u) return q;
    out.vtx_nbr[size_t(fill_n[v]) * n + v] = u;
    return fill_n[v]++;
  };
  out.vtx_w.assign(size_t(vmax + 1) * n, 0.0);
  for (int t = 0; t < T; ++t) {
    const double a = out.tri_rest[4 * t], b = out.tri_rest[4 * t + 1], c = out.tri_rest[4 * t + 2];
    const double A0 = out.tri_rest[4 * t + 3];
    // G = [[-1,-1],[1,0],[0,1]] Dm^-1  (3x2)
    const double G[3][2] = {{-a, -b - c}, {a, b}, {0.0, c}};
    for (int p = 0; p < 3; ++p) {
      const int vp = out.tri[4 * t + p];
      out.vtx_corner[size_t(fill_c[vp]++) * n + vp] = 3 * t + p;
      for (int q = 0; q < 3; ++q) {
        const double w = A0 * (G[p][0] * G[q][0] + G[p][1] * G[q][1]);
        if (p == q) {
          out.vtx_w[vp] += w;
        } else {
          const int slot = nbr_slot(vp, out.tri[4 * t + q]);
          out.vtx_w[size_t(slot + 1) * n + vp] += w;
        }
      }
    }
  }

  // ---- lumped mass (R10) and dense H~ ----------------------------------------------------
  out.mass.resize(n);
  for (int v = 0; v < n; ++v) out.mass[v] = m.density * V0 * out.area_v[v] / A;
  const double k_mem = m.skalak_B + 2.0 * m.skalak_C;
  const double c_mass = (1.0 + h * m.rayleigh_alpha) / (h * h);
  const double c_L = 1.0 + m.rayleigh_beta / h;            // H~ = c_mass M + c_L L
  out.H.assign(size_t(n) * n, 0.0);
  // sparse row p of L_cot as (index, weight) pairs
  auto row = [&](int p, int *idx, double *w) -> int {
    int cnt = 0;
    idx[cnt] = p;
    w[cnt++] = out.vtx_w[p];
    for (int q = 0; q < fill_n[p]; ++q) {
      idx[cnt] = out.vtx_nbr[size_t(q) * n + p];
      w[cnt++] = out.vtx_w[size_t(q + 1) * n + p];
    }
    return cnt;
  };
  int idx[40];
  double w[40];
  for (int p = 0; p < n; ++p) {
    const int cnt = row(p, idx, w);
    out.H[size_t(p) * n + p] += c_mass * out.mass[p];
    for (int i = 0; i < cnt; ++i) {
      out.H[size_t(p) * n + idx[i]] += c_L * k_mem * w[i];                 // k_mem L_cot
      // k_b L_cot^T diag(1/A_v) L_cot: row p of L_cot contributes w_i w_j / A_p to (idx_i, idx_j)
      for (int j = 0; j < cnt; ++j)
        out.H[size_t(idx[i]) * n + idx[j]] += c_L * m.k_bending * w[i] * w[j] / out.area_v[p];
    }
  }
  return NPFEM_OK;
}

}  // namespace npfem
