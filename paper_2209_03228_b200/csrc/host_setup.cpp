// host_setup.cpp -- see host_setup.hpp.  Quadtree cells are addressed by (level, i, j); hanging faces are found
// by neighbour look-up (a face whose neighbour region is covered by a coarser leaf), not by geometry sweeps.
#include "host_setup.hpp"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <map>
#include <string>
#include <tuple>
#include <tuple>
#include <unordered_map>

namespace landau {

namespace {

// Lagrange basis on k+1 equispaced nodes of [-1,1] (reading A9): values and derivatives at x.
void equispaced_lagrange(int k, double x, double* v, double* d) {
  // first-form barycentric-free evaluation with exact integer denominators: nodes t_c = (2c - k)/k
  for (int c = 0; c <= k; ++c) {
    double num = 1.0, den = 1.0;
    for (int j = 0; j <= k; ++j) {
      if (j == c) continue;
      num *= (k * x - (2 * j - k));
      den *= 2.0 * (c - j);
    }
    v[c] = num / den;
    double acc = 0.0;
    for (int skip = 0; skip <= k; ++skip) {
      if (skip == c) continue;
      double p = k;  // d/dx of (k x - (2 skip - k))
      for (int j = 0; j <= k; ++j) {
        if (j == c || j == skip) continue;
        p *= (k * x - (2 * j - k));
      }
      acc += p;
    }
    d[c] = acc / den;
  }
}

struct CellId {
  int level, i, j;
  bool operator<(const CellId& o) const { return std::tie(level, i, j) < std::tie(o.level, o.i, o.j); }
};

}  // namespace

bool build_tables(int k, HostTables* t, std::string* msg) {
  if (k < 2 || k > 4) {
    *msg = "element degree must be 2, 3 or 4";
    return false;
  }
  t->k = k;
  t->nq1 = k + 1;
  t->nb = (k + 1) * (k + 1);
  t->nq = t->nb;
  // closed-form Gauss-Legendre rules
  if (k == 2) {
    const double a = std::sqrt(3.0 / 5.0);
    t->gauss_x = {-a, 0.0, a};
    t->gauss_w = {5.0 / 9.0, 8.0 / 9.0, 5.0 / 9.0};
  } else if (k == 3) {
    const double s = std::sqrt(6.0 / 5.0);
    const double a = std::sqrt(3.0 / 7.0 - 2.0 / 7.0 * s), b = std::sqrt(3.0 / 7.0 + 2.0 / 7.0 * s);
    const double wa = (18.0 + std::sqrt(30.0)) / 36.0, wb = (18.0 - std::sqrt(30.0)) / 36.0;
    t->gauss_x = {-b, -a, a, b};
    t->gauss_w = {wb, wa, wa, wb};
  } else {
    const double s = 2.0 * std::sqrt(10.0 / 7.0);
    const double a = std::sqrt(5.0 - s) / 3.0, b = std::sqrt(5.0 + s) / 3.0;
    const double wa = (322.0 + 13.0 * std::sqrt(70.0)) / 900.0, wb = (322.0 - 13.0 * std::sqrt(70.0)) / 900.0;
    t->gauss_x = {-b, -a, 0.0, a, b};
    t->gauss_w = {wb, wa, 128.0 / 225.0, wa, wb};
  }
  const int n1 = k + 1;
  std::vector<double> v(n1 * n1), d(n1 * n1);  // [q1][c]
  for (int q = 0; q < n1; ++q) equispaced_lagrange(k, t->gauss_x[q], &v[q * n1], &d[q * n1]);
  t->lag_v = v;
  t->lag_d = d;
  t->k3_frag.assign(16 * 32, 0.0);
  if (k <= 3) {  // the ring kernel's fragment tables hold up to 4 x 4 one-dimensional products: Q2 and Q3 only
    // 1-D product tables P[x][y][ac][q] = l^(x)_a(q) l^(y)_c(q), ac = a n1 + c  (zero outside the valid range)
    auto P = [&](int x, int y, int ac, int q) -> double {
      if (ac >= n1 * n1 || q >= n1) return 0.0;
      const int a = ac / n1, c = ac % n1;
      return (x ? d[q * n1 + a] : v[q * n1 + a]) * (y ? d[q * n1 + c] : v[q * n1 + c]);
    };
    // table order used by both directions: 0: P00, 1: P11, 2: P10 (derivative on the test function a), 3: P01
    const int tx[4] = {0, 1, 1, 0}, ty[4] = {0, 1, 0, 1};
    for (int lane = 0; lane < 32; ++lane) {
      const int g = lane >> 2, tq = lane & 3;
      for (int zt = 0; zt < 4; ++zt)
        for (int mt = 0; mt < 2; ++mt)  // stage 1: A[m = a2c2][k = q2]
          t->k3_frag[(zt * 2 + mt) * 32 + lane] = P(tx[zt], ty[zt], g + 8 * mt, tq);
      for (int nt = 0; nt < 2; ++nt)
        for (int h = 0; h < 2; ++h)
          for (int mt = 0; mt < 2; ++mt) {  // stage 2: A[m = a1c1][k -> (rtab = 2 nt + tq/2, q1 = 2 (tq%2) + h)]
            const int rt = 2 * nt + (tq >> 1), q1 = 2 * (tq & 1) + h;
            t->k3_frag[(8 + (nt * 2 + h) * 2 + mt) * 32 + lane] = P(tx[rt], ty[rt], g + 8 * mt, q1);
          }
    }
  }
  t->B.assign(t->nq * t->nb, 0.0);
  t->dBxi.assign(t->nq * t->nb, 0.0);
  t->dBeta.assign(t->nq * t->nb, 0.0);
  for (int q2 = 0; q2 < n1; ++q2)
    for (int q1 = 0; q1 < n1; ++q1)
      for (int a2 = 0; a2 < n1; ++a2)
        for (int a1 = 0; a1 < n1; ++a1) {
          const int q = q1 + n1 * q2, a = a1 + n1 * a2;
          t->B[q * t->nb + a] = v[q1 * n1 + a1] * v[q2 * n1 + a2];
          t->dBxi[q * t->nb + a] = d[q1 * n1 + a1] * v[q2 * n1 + a2];
          t->dBeta[q * t->nb + a] = v[q1 * n1 + a1] * d[q2 * n1 + a2];
        }
  return true;
}

bool build_tables_simplex(int k, HostTables* t, std::string* msg) {
  if (k < 2 || k > 4) {
    *msg = "triangle degree must be 2, 3 or 4";
    return false;
  }
  t->k = k;
  t->nq1 = 0;
  t->simplex = true;
  t->nb = (k + 1) * (k + 2) / 2;
  t->sx.clear();
  t->se.clear();
  t->sw.clear();
  // symmetric rules on the reference triangle, barycentric orbits (a, a, 1 - 2a) and (a, b, 1 - a - b); weights sum to 1/2
  struct Orbit {
    int n;
    double a, b, w;
  };
  static const Orbit deg4[] = {{3, 0.445948490915965, 0, 0.223381589678011}, {3, 0.091576213509771, 0, 0.109951743655322}};
  static const Orbit deg6[] = {{3, 0.249286745170910, 0, 0.116786275726379},
                               {3, 0.063089014491502, 0, 0.050844906370207},
                               {6, 0.053145049844817, 0.310352451033784, 0.082851075618374}};
  static const Orbit deg8[] = {{1, 1.0 / 3.0, 0, 0.144315607677787},
                               {3, 0.459292588292723, 0, 0.095091634267285},
                               {3, 0.170569307751760, 0, 0.103217370534718},
                               {3, 0.050547228317031, 0, 0.032458497623198},
                               {6, 0.008394777409958, 0.263112829634638, 0.027230314174435}};
  const Orbit* rule = k == 2 ? deg4 : k == 3 ? deg6 : deg8;
  const int n_orbits = k == 2 ? 2 : k == 3 ? 3 : 5;
  for (int o = 0; o < n_orbits; ++o) {
    const Orbit& r = rule[o];
    const double c3 = 1.0 - 2.0 * r.a, c6 = 1.0 - r.a - r.b;
    // the orbit's points (lambda_1, lambda_2) = (xi, eta): 1 (centroid), 3 ((a, a, c) permuted) or 6 ((a, b, c) permuted)
    const double p1[1][2] = {{r.a, r.a}};
    const double p3[3][2] = {{r.a, r.a}, {r.a, c3}, {c3, r.a}};
    const double p6[6][2] = {{r.a, r.b}, {r.b, r.a}, {r.a, c6}, {c6, r.a}, {r.b, c6}, {c6, r.b}};
    const double(*pts)[2] = r.n == 1 ? p1 : r.n == 3 ? p3 : p6;
    for (int p = 0; p < r.n; ++p) {
      t->sx.push_back(pts[p][0]);
      t->se.push_back(pts[p][1]);
      t->sw.push_back(0.5 * r.w);
    }
  }
  t->nq = (int)t->sw.size();
  // Lagrange basis of the lattice node (i, j, l = k - i - j): product over the three barycentric coordinates of
  // N_n(lambda) = prod_{m < n} (k lambda - m) / (m + 1); local order j-major, i fastest
  auto factor = [&](int n, double lam, double* v, double* d) {
    double val = 1.0, der = 0.0;
    for (int m = 0; m < n; ++m) {
      const double f = (k * lam - m) / (m + 1.0);
      der = der * f + val * (k / (m + 1.0));
      val *= f;
    }
    *v = val;
    *d = der;
  };
  t->B.assign((size_t)t->nq * t->nb, 0.0);
  t->dBxi.assign((size_t)t->nq * t->nb, 0.0);
  t->dBeta.assign((size_t)t->nq * t->nb, 0.0);
  for (int q = 0; q < t->nq; ++q) {
    const double xi = t->sx[q], eta = t->se[q], lam0 = 1.0 - xi - eta;
    int a = 0;
    for (int j = 0; j <= k; ++j)
      for (int i = 0; i <= k - j; ++i, ++a) {
        double vi, di, vj, dj, vl, dl;
        factor(i, xi, &vi, &di);
        factor(j, eta, &vj, &dj);
        factor(k - i - j, lam0, &vl, &dl);
        t->B[(size_t)q * t->nb + a] = vi * vj * vl;
        t->dBxi[(size_t)q * t->nb + a] = di * vj * vl - vi * vj * dl;   // d lam0 / d xi = -1
        t->dBeta[(size_t)q * t->nb + a] = vi * dj * vl - vi * vj * dl;
      }
  }
  return true;
}

int build_grid(const landau_grid_desc& d, const HostTables& t, HostGrid* g, std::string* msg) {
  if (d.kind != 0 && d.kind != 1) {
    *msg = "grid kind must be 0 (uniform) or 1 (quadtree)";
    return LANDAU_UNSUPPORTED;
  }
  if (!(d.r_max > 0) || !(d.z_max > d.z_min) || d.nr < 1 || d.nz < 1 || (d.kind == 1 && (d.levels < 0 || d.levels > 12))) {
    *msg = "bad grid extents or cell counts";
    return LANDAU_INVALID_ARG;
  }
  const int k = t.k, n1 = k + 1, nb = t.nb, nq = t.nq;
  const int L = d.kind == 1 ? d.levels : 0;
  g->desc = d;
  g->k = k;
  g->nb = nb;
  g->nq = nq;

  // ---- leaves of the quadtree -------------------------------------------------------------------------
  std::vector<CellId> leaves;
  for (int j = 0; j < d.nz; ++j)
    for (int i = 0; i < d.nr; ++i) leaves.push_back(CellId{0, i, j});
  for (int l = 1; l <= L; ++l) {
    std::vector<CellId> next;
    const long long zspan = (long long)d.nz << l;  // 4 x (z centre in level-(l-1) cells) = 4 nz 2^(l-2)
    for (const CellId& c : leaves) {
      // cell (l-1, i, j) in units of level-(l-1) cells; box: r <= nr/2, z in [nz 2^(l-2) -+ nz/4]; times 4:
      bool inside = c.level == l - 1 && 2LL * (c.i + 1) <= d.nr && 4LL * c.j >= zspan - d.nz &&
                    4LL * (c.j + 1) <= zspan + d.nz;
      if (!inside) {
        next.push_back(c);
        continue;
      }
      for (int cj = 0; cj < 2; ++cj)
        for (int ci = 0; ci < 2; ++ci) next.push_back(CellId{l, 2 * c.i + ci, 2 * c.j + cj});
    }
    leaves.swap(next);
  }
  std::map<CellId, int> leaf_index;
  for (size_t e = 0; e < leaves.size(); ++e) leaf_index[leaves[e]] = (int)e;
  g->n_cells = (int)leaves.size();

  // ---- lattice nodes: X = (i k + a1) 2^(L-level), Z likewise; key = Z * XW + X (sorted = z-major order) ----
  const long long XW = ((long long)d.nr * k << L) + 1;
  auto node_key = [&](const CellId& c, int a1, int a2) {
    const long long X = ((long long)c.i * k + a1) << (L - c.level);
    const long long Z = ((long long)c.j * k + a2) << (L - c.level);
    return Z * XW + X;
  };
  // ---- hanging faces: constraint[key] = list of (master key, weight) ------------------------------------
  std::unordered_map<long long, std::vector<std::pair<long long, double>>> constraint;
  std::vector<double> lv(n1), ld(n1);
  for (const CellId& c : leaves) {
    for (int face = 0; face < 4; ++face) {  // 0: r-low, 1: r-high, 2: z-low, 3: z-high
      int ni = c.i + (face == 0 ? -1 : face == 1 ? 1 : 0);
      int nj = c.j + (face == 2 ? -1 : face == 3 ? 1 : 0);
      if (ni < 0 || nj < 0 || ni >= (d.nr << c.level) || nj >= (d.nz << c.level)) continue;  // domain boundary
      // the leaf covering the neighbour position is the neighbour itself (conforming), one of its ancestors
      // (coarser: this face hangs), or neither (neighbour refined further: the finer side owns the constraint)
      CellId nb_cell{c.level, ni, nj};
      bool found = false;
      for (int lev = c.level; lev >= 0; --lev) {
        nb_cell = CellId{lev, ni >> (c.level - lev), nj >> (c.level - lev)};
        if (leaf_index.count(nb_cell)) {
          found = true;
          break;
        }
      }
      if (!found || nb_cell.level == c.level) continue;
      // the face of c lies on an edge of the coarser leaf nb_cell: constrain c's face nodes that are not
      // nodes of nb_cell to the k+1 nodes of that coarse edge
      const int shift = c.level - nb_cell.level;
      const bool along_z = face < 2;  // r-faces run along z
      for (int a = 0; a <= k; ++a) {
        const int a1 = along_z ? (face == 0 ? 0 : k) : a;
        const int a2 = along_z ? a : (face == 2 ? 0 : k);
        // position of the node along the coarse edge, in units of (coarse node spacing / 2^shift)
        const long long fine_pos = along_z ? ((long long)c.j * k + a2) : ((long long)c.i * k + a1);
        const long long coarse_org = (along_z ? (long long)nb_cell.j : (long long)nb_cell.i) * k << shift;
        const long long rel = fine_pos - coarse_org;  // in [0, k 2^shift]
        if (rel % (1LL << shift) == 0) continue;       // coincides with a coarse node
        const double x = -1.0 + 2.0 * (double)rel / (double)((long long)k << shift);
        equispaced_lagrange(k, x, lv.data(), ld.data());
        std::vector<std::pair<long long, double>> row;
        for (int cidx = 0; cidx <= k; ++cidx) {
          // coarse edge node: on the coarse cell's face opposite to `face`
          const int b1 = along_z ? (face == 0 ? k : 0) : cidx;
          const int b2 = along_z ? cidx : (face == 2 ? k : 0);
          row.push_back(std::make_pair(node_key(nb_cell, b1, b2), lv[cidx]));
        }
        constraint[node_key(c, a1, a2)] = row;
      }
    }
  }
  // ---- free nodes -> dofs in (z, r) order ---------------------------------------------------------------------
  std::vector<long long> keys;
  keys.reserve(leaves.size() * nb);
  for (const CellId& c : leaves)
    for (int a2 = 0; a2 <= k; ++a2)
      for (int a1 = 0; a1 <= k; ++a1) {
        long long key = node_key(c, a1, a2);
        if (!constraint.count(key)) keys.push_back(key);
      }
  std::sort(keys.begin(), keys.end());
  keys.erase(std::unique(keys.begin(), keys.end()), keys.end());
  g->n_dof = (int)keys.size();
  std::unordered_map<long long, int> dof_of;
  dof_of.reserve(keys.size() * 2);
  const double ur = d.r_max / (double)((long long)d.nr * k << L);
  const double uz = (d.z_max - d.z_min) / (double)((long long)d.nz * k << L);
  g->dof_r.resize(g->n_dof);
  g->dof_z.resize(g->n_dof);
  for (int n = 0; n < g->n_dof; ++n) {
    dof_of[keys[n]] = n;
    g->dof_r[n] = (double)(keys[n] % XW) * ur;
    g->dof_z[n] = d.z_min + (double)(keys[n] / XW) * uz;
  }
  // ---- rows of P_e -------------------------------------------------------------------------------------------
  g->en_ptr.assign(1, 0);
  g->en_dof.clear();
  g->en_w.clear();
  bool chain_error = false;
  std::vector<std::pair<long long, double>> work, nxt;
  for (const CellId& c : leaves)
    for (int a2 = 0; a2 <= k; ++a2)
      for (int a1 = 0; a1 <= k; ++a1) {
        work.assign(1, std::make_pair(node_key(c, a1, a2), 1.0));
        for (int depth = 0; depth < 6; ++depth) {
          bool again = false;
          nxt.clear();
          for (auto& kw : work) {
            auto it = constraint.find(kw.first);
            if (it == constraint.end()) {
              nxt.push_back(kw);
              continue;
            }
            again = true;
            for (auto& mw : it->second) nxt.push_back(std::make_pair(mw.first, kw.second * mw.second));
          }
          work.swap(nxt);
          if (!again) break;
          if (depth == 5) chain_error = true;
        }
        std::map<int, double> merged;
        for (auto& kw : work) {
          auto it = dof_of.find(kw.first);
          if (it == dof_of.end()) {
            chain_error = true;
            continue;
          }
          merged[it->second] += kw.second;
        }
        for (auto& dw : merged)
          if (dw.second != 0.0) {
            g->en_dof.push_back(dw.first);
            g->en_w.push_back(dw.second);
          }
        g->en_ptr.push_back((int)g->en_dof.size());
      }
  if (chain_error) {
    *msg = "unresolvable hanging-node constraints (mesh not 2:1 balanced)";
    return LANDAU_UNSUPPORTED;
  }
  // ---- cell rectangles and integration points ----------------------------------------------------------------
  g->cell_r0.resize(g->n_cells);
  g->cell_z0.resize(g->n_cells);
  g->cell_hr.resize(g->n_cells);
  g->cell_hz.resize(g->n_cells);
  g->n_ip = g->n_cells * nq;
  g->ip_r.resize(g->n_ip);
  g->ip_z.resize(g->n_ip);
  g->ip_w.resize(g->n_ip);
  for (int e = 0; e < g->n_cells; ++e) {
    const CellId& c = leaves[e];
    const double hr = d.r_max / (double)((long long)d.nr << c.level);
    const double hz = (d.z_max - d.z_min) / (double)((long long)d.nz << c.level);
    g->cell_hr[e] = hr;
    g->cell_hz[e] = hz;
    g->cell_r0[e] = c.i * hr;
    g->cell_z0[e] = d.z_min + c.j * hz;
    for (int q2 = 0; q2 < n1; ++q2)
      for (int q1 = 0; q1 < n1; ++q1) {
        const int ip = e * nq + q1 + n1 * q2;
        const double r = g->cell_r0[e] + 0.5 * hr * (1.0 + t.gauss_x[q1]);
        g->ip_r[ip] = r;
        g->ip_z[ip] = g->cell_z0[e] + 0.5 * hz * (1.0 + t.gauss_x[q2]);
        g->ip_w[ip] = t.gauss_w[q1] * t.gauss_w[q2] * 0.25 * hr * hz * r;
      }
  }
  return finish_grid(t, g, msg);
}

// Everything that follows from the rows of P_e (en_ptr / en_dof / en_w): CSR pattern, assembly and apply gather tables,
// the K3 ring schedule.  Shared by the rectangular / quadtree grids and the unstructured meshes.
int finish_grid(const HostTables& t, HostGrid* g, std::string* msg) {
  (void)msg;
  const int k = t.k, n1 = k + 1, nb = t.nb;
  (void)k;
  // ---- CSR pattern ----------------------------------------------------------------------------------------------
  std::vector<std::vector<int>> rows(g->n_dof);
  std::vector<int> touched;
  for (int e = 0; e < g->n_cells; ++e) {
    touched.assign(g->en_dof.begin() + g->en_ptr[e * nb], g->en_dof.begin() + g->en_ptr[(e + 1) * nb]);
    std::sort(touched.begin(), touched.end());
    touched.erase(std::unique(touched.begin(), touched.end()), touched.end());
    for (int I : touched) rows[I].insert(rows[I].end(), touched.begin(), touched.end());
  }
  g->rowptr.assign(g->n_dof + 1, 0);
  g->colidx.clear();
  for (int I = 0; I < g->n_dof; ++I) {
    std::sort(rows[I].begin(), rows[I].end());
    rows[I].erase(std::unique(rows[I].begin(), rows[I].end()), rows[I].end());
    g->colidx.insert(g->colidx.end(), rows[I].begin(), rows[I].end());
    g->rowptr[I + 1] = (int)g->colidx.size();
  }
  g->nnz = (int)g->colidx.size();
  g->diag.resize(g->n_dof);
  for (int I = 0; I < g->n_dof; ++I)
    g->diag[I] = (int)(std::lower_bound(g->colidx.begin() + g->rowptr[I], g->colidx.begin() + g->rowptr[I + 1], I) -
                       g->colidx.begin());
  // ---- gather tables -----------------------------------------------------------------------------------------------
  {
    std::vector<int> count(g->nnz, 0);
    struct Entry {
      int slot, code;
      double w;
    };
    std::vector<Entry> entries;
    for (int e = 0; e < g->n_cells; ++e)
      for (int a = 0; a < nb; ++a)
        for (int pa = g->en_ptr[e * nb + a]; pa < g->en_ptr[e * nb + a + 1]; ++pa) {
          const int I = g->en_dof[pa];
          const int* rb = &g->colidx[g->rowptr[I]];
          const int* re = rb + (g->rowptr[I + 1] - g->rowptr[I]);
          for (int c = 0; c < nb; ++c)
            for (int pc = g->en_ptr[e * nb + c]; pc < g->en_ptr[e * nb + c + 1]; ++pc) {
              const int slot = (int)(std::lower_bound(rb, re, g->en_dof[pc]) - &g->colidx[0]);
              entries.push_back(Entry{slot, (e * nb + a) * nb + c, g->en_w[pa] * g->en_w[pc]});
              ++count[slot];
            }
        }
    g->as_ptr.assign(g->nnz + 1, 0);
    for (int n = 0; n < g->nnz; ++n) g->as_ptr[n + 1] = g->as_ptr[n] + count[n];
    g->as_code.resize(entries.size());
    g->as_w.resize(entries.size());
    std::vector<int> fill(g->as_ptr.begin(), g->as_ptr.end() - 1);
    for (const Entry& en : entries) {  // entries are generated in (cell, a, c) order => deterministic lists
      g->as_code[fill[en.slot]] = en.code;
      g->as_w[fill[en.slot]] = en.w;
      ++fill[en.slot];
    }
  }
  // ---- K3 ring schedule (tensor-product cells only: the ring kernel is sum-factorised) ----------------------------------
  if (!t.simplex && t.k <= 3) {
    const int nb2 = nb * nb;
    g->k3_nsteps = (g->n_cells + K3_PC - 1) / K3_PC;
    // emission step of every CSR slot = step of its last contributing cell; an element matrix stays in the ring from
    // the step that computes it to the last step that emits one of its slots
    std::vector<int> last(g->nnz, 0), dies(g->n_cells, 0);
    for (int c = 0; c < g->n_cells; ++c) dies[c] = c / K3_PC;
    for (int n = 0; n < g->nnz; ++n) {
      int hi = -1;
      for (int p = g->as_ptr[n]; p < g->as_ptr[n + 1]; ++p) hi = std::max(hi, g->as_code[p] / nb2);
      last[n] = hi;
      for (int p = g->as_ptr[n]; p < g->as_ptr[n + 1]; ++p) {
        int& d = dies[g->as_code[p] / nb2];
        d = std::max(d, hi / K3_PC);
      }
    }
    // ring positions: a cell takes the lowest free position when its step starts; positions of matrices whose last
    // emission was an earlier step are free again (the kernel's second barrier of a step orders reuse after emission)
    g->cell_pos.assign(g->n_cells, 0);
    g->halo_begin.assign(g->k3_nsteps, 0);
    int rc = 0;
    {
      std::vector<int> free_pos, owner;  // owner[pos] = cell or -1
      for (int st = 0; st < g->k3_nsteps; ++st) {
        int hb = st;
        for (size_t pos = 0; pos < owner.size(); ++pos)
          if (owner[pos] >= 0) {
            if (dies[owner[pos]] < st)
              owner[pos] = -1;
            else
              hb = std::min(hb, owner[pos] / K3_PC);
          }
        g->halo_begin[st] = hb;
        for (int c = st * K3_PC; c < std::min(g->n_cells, (st + 1) * K3_PC); ++c) {
          size_t pos = 0;
          while (pos < owner.size() && owner[pos] >= 0) ++pos;
          if (pos == owner.size()) owner.push_back(-1);
          owner[pos] = c;
          g->cell_pos[c] = (int)pos;
        }
        rc = std::max(rc, (int)owner.size());
      }
    }
    if ((long long)rc * K3_RS * 8 + 64 > K3_RING_MAX_BYTES || (long long)rc * K3_RS + 8 >= (1 << (32 - K3_NBITS))) rc = 0;
    g->k3_rc = rc;
    if (rc) {
      const int S1 = g->k3_nsteps + 1;
      g->as_roff.resize(g->as_code.size());
      for (size_t p = 0; p < g->as_code.size(); ++p) {
        const int code = g->as_code[p], cell = code / nb2, a = (code / nb) % nb, c = code % nb;
        const int a1 = a % n1, a2 = a / n1, c1 = c % n1, c2 = c / n1;
        g->as_roff[p] = g->cell_pos[cell] * K3_RS + k3_entry_offset(a2 * n1 + c2, a1 * n1 + c1);
      }
      // classify, bucket by step (slots visited in ascending n, so every list is ascending)
      std::vector<std::vector<int>> l1(g->k3_nsteps), l4(g->k3_nsteps), lg(g->k3_nsteps);
      for (int n = 0; n < g->nnz; ++n) {
        const int p0 = g->as_ptr[n], cnt = g->as_ptr[n + 1] - p0;
        bool unit = cnt <= 4;
        for (int p = p0; p < p0 + cnt && unit; ++p) unit = g->as_w[p] == 1.0;
        (unit ? (cnt == 1 ? l1 : l4) : lg)[last[n] / K3_PC].push_back(n);
      }
      g->em_ptr.assign(3 * S1, 0);
      g->em_base.assign(g->k3_nsteps, 0);
      g->em1.clear();
      g->em4.clear();
      g->emg.clear();
      const unsigned zero_off = (unsigned)(rc * K3_RS);
      for (int st = 0; st < g->k3_nsteps && rc; ++st) {
        int base = g->nnz;
        for (const auto* l : {&l1[st], &l4[st], &lg[st]})
          if (!l->empty()) base = std::min(base, l->front());
        g->em_base[st] = base;
        g->em_ptr[st] = (int)g->em1.size();
        g->em_ptr[S1 + st] = (int)g->em4.size() / 4;
        g->em_ptr[2 * S1 + st] = (int)g->emg.size();
        for (int n : l1[st]) {
          if (n - base >= (1 << K3_NBITS)) rc = 0;
          g->em1.push_back((unsigned)g->as_roff[g->as_ptr[n]] << K3_NBITS | (unsigned)(n - base));
        }
        for (int n : l4[st]) {
          unsigned off[4] = {zero_off, zero_off, zero_off, zero_off};
          for (int p = g->as_ptr[n]; p < g->as_ptr[n + 1]; ++p) off[p - g->as_ptr[n]] = (unsigned)g->as_roff[p];
          g->em4.push_back((unsigned)(n - base));
          g->em4.push_back(off[0] | off[1] << 16);
          g->em4.push_back(off[2] | off[3] << 16);
          g->em4.push_back(0u);
        }
        for (int n : lg[st]) g->emg.push_back(n);
      }
      g->em_ptr[g->k3_nsteps] = (int)g->em1.size();
      g->em_ptr[S1 + g->k3_nsteps] = (int)g->em4.size() / 4;
      g->em_ptr[2 * S1 + g->k3_nsteps] = (int)g->emg.size();
      g->k3_rc = rc;  // 0 if a packed word overflowed
    }
  }
  {
    std::vector<int> count(g->n_dof, 0);
    for (size_t p = 0; p < g->en_dof.size(); ++p) ++count[g->en_dof[p]];
    g->ap_ptr.assign(g->n_dof + 1, 0);
    for (int n = 0; n < g->n_dof; ++n) g->ap_ptr[n + 1] = g->ap_ptr[n] + count[n];
    g->ap_code.resize(g->en_dof.size());
    g->ap_w.resize(g->en_dof.size());
    std::vector<int> fill(g->ap_ptr.begin(), g->ap_ptr.end() - 1);
    for (int ea = 0; ea < g->n_cells * nb; ++ea)
      for (int p = g->en_ptr[ea]; p < g->en_ptr[ea + 1]; ++p) {
        const int I = g->en_dof[p];
        g->ap_code[fill[I]] = ea;
        g->ap_w[fill[I]] = g->en_w[p];
        ++fill[I];
      }
  }
  return LANDAU_OK;
}

// ---- unstructured conforming meshes of straight-sided quadrilaterals (sec. 5.2) -------------------------
// Nodes are identified by topology, not geometry: a corner node by its vertex id, an edge node by (lower vertex id, higher
// vertex id, position counted from the lower one), an interior node by (cell, a1, a2).  Dofs are then ordered by their
// coordinates on a grid of 2^-30 of the mesh extent, z-major.
// triangles: the same topological identification (vertex / edge / interior keys), affine geometry
static int build_triangle_grid(const landau_mesh_desc& m, const HostTables& t, HostGrid* g, std::string* msg) {
  const int k = t.k, nb = t.nb, nq = t.nq, nc = m.n_cells;
  memset(&g->desc, 0, sizeof(g->desc));
  g->desc.kind = 3;
  g->k = k;
  g->nb = nb;
  g->nq = nq;
  g->n_cells = nc;
  for (int e = 0; e < 3 * nc; ++e)
    if (m.cells[e] < 0 || m.cells[e] >= m.n_vertices) {
      *msg = "mesh cell refers to a missing vertex";
      return LANDAU_INVALID_ARG;
    }
  double scale = 0.0;
  for (int v = 0; v < 2 * m.n_vertices; ++v) scale = std::max(scale, std::fabs(m.vertices_rz[v]));
  const double quantum = scale / 1073741824.0;
  typedef std::tuple<int, int, int, int> NodeKey;
  std::map<NodeKey, int> node_of;
  std::vector<double> nr, nz;
  std::vector<int> cell_node((size_t)nc * nb);
  auto edge_key = [&](int va, int vb, int tpos) { return va < vb ? NodeKey(1, va, vb, tpos) : NodeKey(1, vb, va, k - tpos); };
  for (int e = 0; e < nc; ++e) {
    const int* cv = &m.cells[3 * e];
    const double* P0 = &m.vertices_rz[2 * cv[0]];
    const double* P1 = &m.vertices_rz[2 * cv[1]];
    const double* P2 = &m.vertices_rz[2 * cv[2]];
    int a = 0;
    for (int j = 0; j <= k; ++j)
      for (int i = 0; i <= k - j; ++i, ++a) {
        const int l = k - i - j;
        NodeKey key;
        if (i == k)
          key = NodeKey(0, cv[1], 0, 0);
        else if (j == k)
          key = NodeKey(0, cv[2], 0, 0);
        else if (l == k)
          key = NodeKey(0, cv[0], 0, 0);
        else if (j == 0)
          key = edge_key(cv[0], cv[1], i);  // on v0 -> v1, i steps from v0
        else if (l == 0)
          key = edge_key(cv[1], cv[2], j);  // on v1 -> v2, j steps from v1
        else if (i == 0)
          key = edge_key(cv[0], cv[2], j);  // on v0 -> v2, j steps from v0
        else
          key = NodeKey(2, e, i, j);
        auto it = node_of.find(key);
        int id;
        if (it == node_of.end()) {
          id = (int)nr.size();
          node_of[key] = id;
          const double xi = (double)i / k, eta = (double)j / k;
          nr.push_back(P0[0] + (P1[0] - P0[0]) * xi + (P2[0] - P0[0]) * eta);
          nz.push_back(P0[1] + (P1[1] - P0[1]) * xi + (P2[1] - P0[1]) * eta);
        } else {
          id = it->second;
        }
        cell_node[(size_t)e * nb + a] = id;
      }
  }
  const int nn = (int)nr.size();
  std::vector<std::pair<std::pair<long long, long long>, int>> order(nn);
  for (int i = 0; i < nn; ++i) order[i] = std::make_pair(std::make_pair(std::llround(nz[i] / quantum), std::llround(nr[i] / quantum)), i);
  std::sort(order.begin(), order.end());
  std::vector<int> dof_of(nn);
  g->n_dof = nn;
  g->dof_r.resize(nn);
  g->dof_z.resize(nn);
  for (int I = 0; I < nn; ++I) {
    dof_of[order[I].second] = I;
    g->dof_r[I] = nr[order[I].second];
    g->dof_z[I] = nz[order[I].second];
  }
  g->en_ptr.assign(1, 0);
  g->en_dof.clear();
  g->en_w.clear();
  for (int ea = 0; ea < nc * nb; ++ea) {
    g->en_dof.push_back(dof_of[cell_node[ea]]);
    g->en_w.push_back(1.0);
    g->en_ptr.push_back((int)g->en_dof.size());
  }
  g->cell_r0.assign(nc, 0.0);
  g->cell_z0.assign(nc, 0.0);
  g->cell_hr.assign(nc, 2.0);
  g->cell_hz.assign(nc, 2.0);
  g->n_ip = nc * nq;
  g->ip_r.resize(g->n_ip);
  g->ip_z.resize(g->n_ip);
  g->ip_w.resize(g->n_ip);
  g->ip_gm.resize(4 * (size_t)g->n_ip);
  for (int e = 0; e < nc; ++e) {
    const int* cv = &m.cells[3 * e];
    const double* P0 = &m.vertices_rz[2 * cv[0]];
    const double J[4] = {m.vertices_rz[2 * cv[1]] - P0[0], m.vertices_rz[2 * cv[2]] - P0[0], m.vertices_rz[2 * cv[1] + 1] - P0[1],
                         m.vertices_rz[2 * cv[2] + 1] - P0[1]};
    const double det = J[0] * J[3] - J[1] * J[2];
    if (!(det > 0.0)) {
      *msg = "mesh cell " + std::to_string(e) + " is inverted or clockwise";
      return LANDAU_INVALID_ARG;
    }
    for (int q = 0; q < nq; ++q) {
      const int ip = e * nq + q;
      g->ip_r[ip] = P0[0] + J[0] * t.sx[q] + J[1] * t.se[q];
      g->ip_z[ip] = P0[1] + J[2] * t.sx[q] + J[3] * t.se[q];
      g->ip_w[ip] = t.sw[q] * det * g->ip_r[ip];
      g->ip_gm[4 * (size_t)ip] = J[3] / det;
      g->ip_gm[4 * (size_t)ip + 1] = -J[2] / det;
      g->ip_gm[4 * (size_t)ip + 2] = -J[1] / det;
      g->ip_gm[4 * (size_t)ip + 3] = J[0] / det;
    }
  }
  return finish_grid(t, g, msg);
}

int build_mesh_grid(const landau_mesh_desc& m, const HostTables& t, HostGrid* g, std::string* msg) {
  if (m.n_vertices < 3 || m.n_cells < 1 || !m.vertices_rz || !m.cells) {
    *msg = "bad mesh: at least one cell and its vertices";
    return LANDAU_INVALID_ARG;
  }
  if ((m.vertices_per_cell == 3) != t.simplex || (m.vertices_per_cell != 3 && m.vertices_per_cell != 4)) {
    *msg = "mesh cell type does not match the context's element tables (all meshes must have the same vertices_per_cell, 3 or 4)";
    return LANDAU_UNSUPPORTED;
  }
  if (m.n_vertices < m.vertices_per_cell) {
    *msg = "bad mesh: fewer vertices than one cell has";
    return LANDAU_INVALID_ARG;
  }
  {  // the dof ordering divides by 2^-30 of the largest coordinate: it must be finite and non-zero
    double extent = 0.0;
    for (int v = 0; v < 2 * m.n_vertices; ++v) {
      if (!std::isfinite(m.vertices_rz[v])) {
        *msg = "bad mesh: vertex coordinate " + std::to_string(v) + " is not finite";
        return LANDAU_INVALID_ARG;
      }
      extent = std::max(extent, std::fabs(m.vertices_rz[v]));
    }
    if (!(extent > 0.0)) {
      *msg = "bad mesh: every vertex coordinate is zero";
      return LANDAU_INVALID_ARG;
    }
  }
  if (t.simplex) return build_triangle_grid(m, t, g, msg);
  const int k = t.k, n1 = k + 1, nb = t.nb, nq = t.nq, nc = m.n_cells;
  memset(&g->desc, 0, sizeof(g->desc));
  g->desc.kind = 2;
  g->k = k;
  g->nb = nb;
  g->nq = nq;
  g->n_cells = nc;
  for (int e = 0; e < 4 * nc; ++e)
    if (m.cells[e] < 0 || m.cells[e] >= m.n_vertices) {
      *msg = "mesh cell refers to a missing vertex";
      return LANDAU_INVALID_ARG;
    }
  double scale = 0.0;
  for (int v = 0; v < 2 * m.n_vertices; ++v) scale = std::max(scale, std::fabs(m.vertices_rz[v]));
  const double quantum = scale / 1073741824.0;
  auto vert = [&](int e, int c, int d) { return m.vertices_rz[2 * m.cells[4 * e + c] + d]; };
  // bilinear map of cell e and its Jacobian [dr/dxi, dr/deta, dz/dxi, dz/deta]
  auto map_point = [&](int e, double xi, double eta, double* x, double* J) {
    const double N[4] = {0.25 * (1 - xi) * (1 - eta), 0.25 * (1 + xi) * (1 - eta), 0.25 * (1 + xi) * (1 + eta), 0.25 * (1 - xi) * (1 + eta)};
    const double Nx[4] = {-0.25 * (1 - eta), 0.25 * (1 - eta), 0.25 * (1 + eta), -0.25 * (1 + eta)};
    const double Ne[4] = {-0.25 * (1 - xi), -0.25 * (1 + xi), 0.25 * (1 + xi), 0.25 * (1 - xi)};
    x[0] = x[1] = 0.0;
    if (J) J[0] = J[1] = J[2] = J[3] = 0.0;
    for (int c = 0; c < 4; ++c) {
      x[0] += N[c] * vert(e, c, 0);
      x[1] += N[c] * vert(e, c, 1);
      if (J) {
        J[0] += Nx[c] * vert(e, c, 0);
        J[1] += Ne[c] * vert(e, c, 0);
        J[2] += Nx[c] * vert(e, c, 1);
        J[3] += Ne[c] * vert(e, c, 1);
      }
    }
  };
  typedef std::tuple<int, int, int, int> NodeKey;  // (kind, i, j, l)
  std::map<NodeKey, int> node_of;
  std::vector<double> nr, nz;
  std::vector<int> cell_node((size_t)nc * nb);
  auto edge_key = [&](int va, int vb, int tpos) { return va < vb ? NodeKey(1, va, vb, tpos) : NodeKey(1, vb, va, k - tpos); };
  for (int e = 0; e < nc; ++e) {
    const int* cv = &m.cells[4 * e];
    for (int a2 = 0; a2 <= k; ++a2)
      for (int a1 = 0; a1 <= k; ++a1) {
        NodeKey key;
        const bool x0 = a1 == 0, x1 = a1 == k, y0 = a2 == 0, y1 = a2 == k;
        if ((x0 || x1) && (y0 || y1))
          key = NodeKey(0, cv[y0 ? (x0 ? 0 : 1) : (x0 ? 3 : 2)], 0, 0);
        else if (y0)
          key = edge_key(cv[0], cv[1], a1);
        else if (x1)
          key = edge_key(cv[1], cv[2], a2);
        else if (y1)
          key = edge_key(cv[3], cv[2], a1);
        else if (x0)
          key = edge_key(cv[0], cv[3], a2);
        else
          key = NodeKey(2, e, a1, a2);
        auto it = node_of.find(key);
        int id;
        if (it == node_of.end()) {
          id = (int)nr.size();
          node_of[key] = id;
          double x[2];
          map_point(e, -1.0 + 2.0 * a1 / k, -1.0 + 2.0 * a2 / k, x, nullptr);
          nr.push_back(x[0]);
          nz.push_back(x[1]);
        } else {
          id = it->second;
        }
        cell_node[(size_t)e * nb + a1 + n1 * a2] = id;
      }
  }
  const int nn = (int)nr.size();
  std::vector<std::pair<std::pair<long long, long long>, int>> order(nn);
  for (int i = 0; i < nn; ++i) order[i] = std::make_pair(std::make_pair(std::llround(nz[i] / quantum), std::llround(nr[i] / quantum)), i);
  std::sort(order.begin(), order.end());
  std::vector<int> dof_of(nn);
  g->n_dof = nn;
  g->dof_r.resize(nn);
  g->dof_z.resize(nn);
  for (int I = 0; I < nn; ++I) {
    dof_of[order[I].second] = I;
    g->dof_r[I] = nr[order[I].second];
    g->dof_z[I] = nz[order[I].second];
  }
  g->en_ptr.assign(1, 0);
  g->en_dof.clear();
  g->en_w.clear();
  for (int ea = 0; ea < nc * nb; ++ea) {
    g->en_dof.push_back(dof_of[cell_node[ea]]);
    g->en_w.push_back(1.0);
    g->en_ptr.push_back((int)g->en_dof.size());
  }
  // the kernels work in reference coordinates on these grids: unit scale factors, J^-T per point (ip_gm)
  g->cell_r0.assign(nc, 0.0);
  g->cell_z0.assign(nc, 0.0);
  g->cell_hr.assign(nc, 2.0);
  g->cell_hz.assign(nc, 2.0);
  g->n_ip = nc * nq;
  g->ip_r.resize(g->n_ip);
  g->ip_z.resize(g->n_ip);
  g->ip_w.resize(g->n_ip);
  g->ip_gm.resize(4 * (size_t)g->n_ip);
  for (int e = 0; e < nc; ++e)
    for (int q2 = 0; q2 < n1; ++q2)
      for (int q1 = 0; q1 < n1; ++q1) {
        const int ip = e * nq + q1 + n1 * q2;
        double x[2], J[4];
        map_point(e, t.gauss_x[q1], t.gauss_x[q2], x, J);
        const double det = J[0] * J[3] - J[1] * J[2];
        if (!(det > 0.0)) {
          *msg = "mesh cell " + std::to_string(e) + " is inverted or clockwise";
          return LANDAU_INVALID_ARG;
        }
        g->ip_r[ip] = x[0];
        g->ip_z[ip] = x[1];
        g->ip_w[ip] = t.gauss_w[q1] * t.gauss_w[q2] * det * x[0];
        g->ip_gm[4 * (size_t)ip] = J[3] / det;       // (d/dr, d/dz) = gm (d/dxi, d/deta)
        g->ip_gm[4 * (size_t)ip + 1] = -J[2] / det;
        g->ip_gm[4 * (size_t)ip + 2] = -J[1] / det;
        g->ip_gm[4 * (size_t)ip + 3] = J[0] / det;
      }
  return finish_grid(t, g, msg);
}

}  // namespace landau
