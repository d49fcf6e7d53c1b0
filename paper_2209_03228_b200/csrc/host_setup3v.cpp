// host_setup3v.cpp -- see host_setup3v.hpp.
#include "host_setup3v.hpp"

#include <algorithm>
#include <cmath>
#include <map>
#include <unordered_map>

namespace landau3v {

namespace {

struct Leaf {
  int level, i, j, k;
};

inline unsigned long long leaf_key(int level, long long i, long long j, long long k) {
  return ((unsigned long long)level << 57) | ((unsigned long long)i << 38) | ((unsigned long long)j << 19) | (unsigned long long)k;
}

// quadratic Lagrange polynomials on the nodes 0, 1, 2 of a cell edge, at t in [0, 2] (cell-node units)
inline void quad_weights(double t, double* w) {
  w[0] = 0.5 * (t - 1.0) * (t - 2.0);
  w[1] = t * (2.0 - t);
  w[2] = 0.5 * t * (t - 1.0);
}

}  // namespace

void build_tables3(HostTables3* t) {
  const double a = std::sqrt(0.6);
  t->gauss_x[0] = -a;
  t->gauss_x[1] = 0.0;
  t->gauss_x[2] = a;
  t->gauss_w[0] = t->gauss_w[2] = 5.0 / 9.0;
  t->gauss_w[1] = 8.0 / 9.0;
  double v[3][3], d[3][3];
  for (int q = 0; q < 3; ++q) {
    const double x = t->gauss_x[q];
    v[q][0] = 0.5 * x * (x - 1.0);
    v[q][1] = 1.0 - x * x;
    v[q][2] = 0.5 * x * (x + 1.0);
    d[q][0] = x - 0.5;
    d[q][1] = -2.0 * x;
    d[q][2] = x + 0.5;
  }
  t->B.assign(NQ * NB, 0.0);
  t->dBx.assign(NQ * NB, 0.0);
  t->dBy.assign(NQ * NB, 0.0);
  t->dBz.assign(NQ * NB, 0.0);
  for (int q = 0; q < NQ; ++q)
    for (int a_ = 0; a_ < NB; ++a_) {
      const int q1 = q % 3, q2 = (q / 3) % 3, q3 = q / 9, a1 = a_ % 3, a2 = (a_ / 3) % 3, a3 = a_ / 9;
      t->B[q * NB + a_] = v[q1][a1] * v[q2][a2] * v[q3][a3];
      t->dBx[q * NB + a_] = d[q1][a1] * v[q2][a2] * v[q3][a3];
      t->dBy[q * NB + a_] = v[q1][a1] * d[q2][a2] * v[q3][a3];
      t->dBz[q * NB + a_] = v[q1][a1] * v[q2][a2] * d[q3][a3];
    }
}

int build_grid3(const landau3v_grid_desc& d, const HostTables3& t, HostGrid3* g, std::string* msg) {
  if (!(d.half_width > 0) || d.n < 1 || d.n > 64 || d.levels < 0 || d.levels > 8) {
    *msg = "bad 3V grid: half_width > 0, 1 <= n <= 64, 0 <= levels <= 8";
    return LANDAU_INVALID_ARG;
  }
  g->desc = d;
  const int L = d.levels, n = d.n;
  // ---- leaves: refine, level by level, the cells around the centre (index range [c - 1, c] per direction for even
  //      extents, the single middle cell for odd ones)
  std::vector<Leaf> leaves;
  for (int k = 0; k < n; ++k)
    for (int j = 0; j < n; ++j)
      for (int i = 0; i < n; ++i) leaves.push_back(Leaf{0, i, j, k});
  for (int l = 1; l <= L; ++l) {
    const long long ext = (long long)n << (l - 1);  // cells per direction at level l-1
    const long long lo = ext % 2 == 0 ? ext / 2 - 1 : ext / 2, hi = ext / 2;
    std::vector<Leaf> next;
    for (const Leaf& c : leaves) {
      const bool mid = c.level == l - 1 && c.i >= lo && c.i <= hi && c.j >= lo && c.j <= hi && c.k >= lo && c.k <= hi;
      if (!mid) {
        next.push_back(c);
        continue;
      }
      for (int b = 0; b < 8; ++b) next.push_back(Leaf{l, 2 * c.i + (b & 1), 2 * c.j + ((b >> 1) & 1), 2 * c.k + (b >> 2)});
    }
    leaves.swap(next);
  }
  g->n_cells = (int)leaves.size();
  std::unordered_map<unsigned long long, int> leaf_at;
  leaf_at.reserve(leaves.size() * 2);
  for (size_t e = 0; e < leaves.size(); ++e) leaf_at[leaf_key(leaves[e].level, leaves[e].i, leaves[e].j, leaves[e].k)] = (int)e;

  // ---- lattice: node a of cell (level, i) sits at (2 i + a) 2^(L - level) on a lattice of W points per direction
  const long long W = ((long long)2 * n << L) + 1;
  auto point_key = [&](long long X, long long Y, long long Z) { return (Z * W + Y) * W + X; };
  auto cell_node = [&](const Leaf& c, int a, long long* P) {
    const int sh = L - c.level;
    P[0] = (long long)(2 * c.i + a % 3) << sh;
    P[1] = (long long)(2 * c.j + (a / 3) % 3) << sh;
    P[2] = (long long)(2 * c.k + a / 9) << sh;
  };
  // master[key] = (leaf, weights) for points that hang: among the leaves whose closure holds the point, found level by
  // level through the hash, the coarsest one that does not have the point as a node
  std::unordered_map<long long, int> hanging_on;
  auto find_host = [&](const long long* P) -> int {
    for (int lev = 0; lev <= L; ++lev) {
      const long long cs = 2LL << (L - lev), hs = cs / 2;  // cell edge and node spacing in lattice units
      long long idx[3][2];
      int cnt[3];
      for (int dd = 0; dd < 3; ++dd) {
        cnt[dd] = 0;
        const long long q = P[dd] / cs;
        if (q < ((long long)n << lev)) idx[dd][cnt[dd]++] = q;
        if (P[dd] % cs == 0 && q > 0) idx[dd][cnt[dd]++] = q - 1;
      }
      for (int c3 = 0; c3 < cnt[2]; ++c3)
        for (int c2 = 0; c2 < cnt[1]; ++c2)
          for (int c1 = 0; c1 < cnt[0]; ++c1) {
            auto it = leaf_at.find(leaf_key(lev, idx[0][c1], idx[1][c2], idx[2][c3]));
            if (it == leaf_at.end()) continue;
            const long long o[3] = {idx[0][c1] * cs, idx[1][c2] * cs, idx[2][c3] * cs};
            if ((P[0] - o[0]) % hs || (P[1] - o[1]) % hs || (P[2] - o[2]) % hs) return it->second;
          }
    }
    return -1;
  };
  std::vector<long long> keys;
  keys.reserve(leaves.size() * NB);
  for (const Leaf& c : leaves)
    for (int a = 0; a < NB; ++a) {
      long long P[3];
      cell_node(c, a, P);
      const long long key = point_key(P[0], P[1], P[2]);
      if (hanging_on.count(key)) continue;
      const int host = L > 0 ? find_host(P) : -1;
      if (host >= 0)
        hanging_on[key] = host;
      else
        keys.push_back(key);
    }
  std::sort(keys.begin(), keys.end());
  keys.erase(std::unique(keys.begin(), keys.end()), keys.end());
  g->n_dof = (int)keys.size();
  std::unordered_map<long long, int> dof_of;
  dof_of.reserve(keys.size() * 2);
  const double unit = 2.0 * d.half_width / (double)(W - 1);
  g->dof_xyz.resize(3 * keys.size());
  for (int I = 0; I < g->n_dof; ++I) {
    dof_of[keys[I]] = I;
    g->dof_xyz[3 * I] = -d.half_width + unit * (double)(keys[I] % W);
    g->dof_xyz[3 * I + 1] = -d.half_width + unit * (double)((keys[I] / W) % W);
    g->dof_xyz[3 * I + 2] = -d.half_width + unit * (double)(keys[I] / (W * W));
  }
  // ---- rows of P_e: expand hanging points through their host cell until only dofs remain
  g->en_ptr.assign(1, 0);
  std::vector<std::pair<long long, double>> work, nxt;
  for (const Leaf& c : leaves)
    for (int a = 0; a < NB; ++a) {
      long long P[3];
      cell_node(c, a, P);
      work.assign(1, std::make_pair(point_key(P[0], P[1], P[2]), 1.0));
      for (int depth = 0;; ++depth) {
        bool again = false;
        nxt.clear();
        for (auto& kw : work) {
          auto it = hanging_on.find(kw.first);
          if (it == hanging_on.end()) {
            nxt.push_back(kw);
            continue;
          }
          again = true;
          const Leaf& h = leaves[it->second];
          const long long hs = 1LL << (L - h.level);
          const long long Q[3] = {kw.first % W, (kw.first / W) % W, kw.first / (W * W)};
          const long long o[3] = {(long long)(2 * h.i) * hs, (long long)(2 * h.j) * hs, (long long)(2 * h.k) * hs};
          double w[3][3];
          for (int dd = 0; dd < 3; ++dd) quad_weights((double)(Q[dd] - o[dd]) / (double)hs, w[dd]);
          for (int b = 0; b < NB; ++b) {
            const double wt = w[0][b % 3] * w[1][(b / 3) % 3] * w[2][b / 9];
            if (wt == 0.0) continue;
            long long M[3];
            cell_node(h, b, M);
            nxt.push_back(std::make_pair(point_key(M[0], M[1], M[2]), kw.second * wt));
          }
        }
        work.swap(nxt);
        if (!again) break;
        if (depth == 8) {
          *msg = "unresolvable hanging-node constraints";
          return LANDAU_UNSUPPORTED;
        }
      }
      std::map<int, double> merged;
      for (auto& kw : work) merged[dof_of.at(kw.first)] += kw.second;
      for (auto& dw : merged)
        if (dw.second != 0.0) {
          g->en_dof.push_back(dw.first);
          g->en_w.push_back(dw.second);
        }
      g->en_ptr.push_back((int)g->en_dof.size());
    }
  // ---- cells and integration points
  g->cell_h.resize(g->n_cells);
  g->n_ip = g->n_cells * NQ;
  g->ip_x.resize(g->n_ip);
  g->ip_y.resize(g->n_ip);
  g->ip_z.resize(g->n_ip);
  g->ip_w.resize(g->n_ip);
  for (int e = 0; e < g->n_cells; ++e) {
    const Leaf& c = leaves[e];
    const double h = 2.0 * d.half_width / (double)((long long)n << c.level);
    g->cell_h[e] = h;
    const double o[3] = {-d.half_width + c.i * h, -d.half_width + c.j * h, -d.half_width + c.k * h};
    for (int q = 0; q < NQ; ++q) {
      const int q1 = q % 3, q2 = (q / 3) % 3, q3 = q / 9;
      g->ip_x[e * NQ + q] = o[0] + 0.5 * h * (1.0 + t.gauss_x[q1]);
      g->ip_y[e * NQ + q] = o[1] + 0.5 * h * (1.0 + t.gauss_x[q2]);
      g->ip_z[e * NQ + q] = o[2] + 0.5 * h * (1.0 + t.gauss_x[q3]);
      g->ip_w[e * NQ + q] = t.gauss_w[q1] * t.gauss_w[q2] * t.gauss_w[q3] * 0.125 * h * h * h;
    }
  }
  // ---- CSR pattern (structural: every pair of dofs that meet in a cell)
  {
    std::vector<std::vector<int>> rows(g->n_dof);
    std::vector<int> touched;
    for (int e = 0; e < g->n_cells; ++e) {
      touched.assign(g->en_dof.begin() + g->en_ptr[e * NB], g->en_dof.begin() + g->en_ptr[(e + 1) * NB]);
      std::sort(touched.begin(), touched.end());
      touched.erase(std::unique(touched.begin(), touched.end()), touched.end());
      for (int I : touched) rows[I].insert(rows[I].end(), touched.begin(), touched.end());
    }
    g->rowptr.assign(g->n_dof + 1, 0);
    for (int I = 0; I < g->n_dof; ++I) {
      std::sort(rows[I].begin(), rows[I].end());
      rows[I].erase(std::unique(rows[I].begin(), rows[I].end()), rows[I].end());
      g->colidx.insert(g->colidx.end(), rows[I].begin(), rows[I].end());
      g->rowptr[I + 1] = (int)g->colidx.size();
    }
    g->nnz = (int)g->colidx.size();
    g->diag.resize(g->n_dof);
    for (int I = 0; I < g->n_dof; ++I)
      g->diag[I] = (int)(std::lower_bound(g->colidx.begin() + g->rowptr[I], g->colidx.begin() + g->rowptr[I + 1], I) - g->colidx.begin());
  }
  // ---- gather tables
  {
    std::vector<int> count(g->nnz, 0);
    struct Entry {
      int slot, code;
      double w;
    };
    std::vector<Entry> entries;
    for (int e = 0; e < g->n_cells; ++e)
      for (int a = 0; a < NB; ++a)
        for (int pa = g->en_ptr[e * NB + a]; pa < g->en_ptr[e * NB + a + 1]; ++pa) {
          const int I = g->en_dof[pa];
          const int* rb = &g->colidx[g->rowptr[I]];
          const int* re = &g->colidx[0] + g->rowptr[I + 1];
          for (int c = 0; c < NB; ++c)
            for (int pc = g->en_ptr[e * NB + c]; pc < g->en_ptr[e * NB + c + 1]; ++pc) {
              const int slot = (int)(std::lower_bound(rb, re, g->en_dof[pc]) - &g->colidx[0]);
              entries.push_back(Entry{slot, (e * NB + a) * NB + c, g->en_w[pa] * g->en_w[pc]});
              ++count[slot];
            }
        }
    g->as_ptr.assign(g->nnz + 1, 0);
    for (int s = 0; s < g->nnz; ++s) g->as_ptr[s + 1] = g->as_ptr[s] + count[s];
    g->as_code.resize(entries.size());
    g->as_w.resize(entries.size());
    std::vector<int> fill(g->as_ptr.begin(), g->as_ptr.end() - 1);
    for (const Entry& en : entries) {
      g->as_code[fill[en.slot]] = en.code;
      g->as_w[fill[en.slot]] = en.w;
      ++fill[en.slot];
    }
  }
  {
    std::vector<int> count(g->n_dof, 0);
    for (size_t p = 0; p < g->en_dof.size(); ++p) ++count[g->en_dof[p]];
    g->ap_ptr.assign(g->n_dof + 1, 0);
    for (int I = 0; I < g->n_dof; ++I) g->ap_ptr[I + 1] = g->ap_ptr[I] + count[I];
    g->ap_code.resize(g->en_dof.size());
    g->ap_w.resize(g->en_dof.size());
    std::vector<int> fill(g->ap_ptr.begin(), g->ap_ptr.end() - 1);
    for (int ea = 0; ea < g->n_cells * NB; ++ea)
      for (int p = g->en_ptr[ea]; p < g->en_ptr[ea + 1]; ++p) {
        const int I = g->en_dof[p];
        g->ap_code[fill[I]] = ea;
        g->ap_w[fill[I]] = g->en_w[p];
        ++fill[I];
      }
  }
  return LANDAU_OK;
}

}  // namespace landau3v
