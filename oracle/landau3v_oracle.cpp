// landau3v_oracle.cpp -- TEST INFRASTRUCTURE ONLY (oracle), 3V variant.
//
// Plain, slow CPU restatement of the discrete Landau collision operator of arxiv 2209.03228 ("PAPER.md") in full 3-D
// velocity space (the "3V model" of PAPER.md:92 sec. 2.3, workload of PAPER.md:125, Tables 6, 14, 16), used only by
// tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.  It shares no code, header, table
// or constant with the CUDA product path (paper_2209_03228_b200/csrc/) -- nor with the 2V oracle next to it -- and the
// product never links or calls it.
//
// What it follows (PAPER.md line : passage):
//   * eq. (2.1), PAPER.md:44-48  -- C[fa,fb] = nu_ab (m0/ma) div INT U . ((m0/ma) fb grad fa - (m0/mb) fa grad fb),
//                                   U(v, vb) = (|u|^2 I - u u^T) / |u|^3,  u = v - vb   (the Landau tensor, 3 x 3 symmetric)
//   * eq. (2.3), PAPER.md:59-64  -- D = sum_b INT U fb d^3vb (symmetric 3 x 3),  K = sum_b INT U . grad fb d^3vb (3-vector)
//   * eq. (2.4), PAPER.md:68-71  -- weak form after integration by parts (sign reading A4 of DESIGN.md)
//   * PAPER.md:73, 75-77         -- frozen-coefficient Jacobian, output M/dt - J (readings A5, A15)
//   * PAPER.md:125               -- "4 x 4 x 4 initial grid", "one level of AMR refinement about the origin", "120 (Q2
//                                   elements) in 3V", "1,045 equations with an average of 54.0 non-zeros per row":
//                                   hexahedral Q2 cells on [-L, L]^3, the 8 cells touching the origin refined, nodes
//                                   hanging on coarse faces / edges constrained, no essential boundary conditions
//
// Conventions are those of the 2V oracle where they carry over (DESIGN.md readings): Cartesian weights w = gw gw gw h^3 / 8
// (no 2 pi, no r: nothing is gyro-averaged here), equispaced Lagrange nodes, f_h = nodal interpolant, coincident points
// (|u|^2 <= 1e-20 (|v|^2 + |vb|^2)) contribute zero, nu_ab = q_a^2 q_b^2 unless a matrix is given, m0 = 1.
// Steps O1..O10 as in DESIGN.md, in plain loops; inner sums in long double; OpenMP over field points only.
//
// Parity pins (tests/test_oracle3v_pins.py): tensor identities (U = U^T, U u = 0, trace 2/|u|), the paper's mesh statistics
// (120 cells / 1,045 equations / 54.0 non-zeros per row), mass = volume and polynomial reproduction through hanging
// faces and edges, Rosenbluth closed forms at an exterior point, conservation of density, all three momenta and energy
// to round-off, brute force on tiny grids (with hanging nodes) and the isotropisation rate of PAPER.md App. B at t = 0
// (the same constant as the 2V pin P10: the Cartesian and the gyro-averaged operator share one normalisation).

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef long double ld;

namespace {

const ld PI_L = 3.14159265358979323846264338327950288419716939937510L;
const int K = 2, N1 = 3, NB = 27, NQ = 27;  // Q2 hexahedra, 3 x 3 x 3 Gauss points (Table 13: (k+1)^d points)

// O1: 3-point Gauss-Legendre on [-1,1], closed form
const ld GX[3] = {-0.774596669241483377035853079956479922L, 0.0L, 0.774596669241483377035853079956479922L};
const ld GW[3] = {5.0L / 9.0L, 8.0L / 9.0L, 5.0L / 9.0L};

// O2: quadratic Lagrange basis on the nodes -1, 0, 1
void lagrange2(ld x, ld* v, ld* d) {
  v[0] = x * (x - 1) / 2;
  v[1] = (1 - x) * (1 + x);
  v[2] = x * (x + 1) / 2;
  d[0] = x - 0.5L;
  d[1] = -2 * x;
  d[2] = x + 0.5L;
}

struct Grid3 {
  double half;
  int n, levels;
  int n_cells = 0, n_dof = 0, n_ip = 0, nnz = 0;
  std::vector<int> lev, ci, cj, ck;      // leaves
  std::vector<double> cx0, cy0, cz0, ch;  // cell origin and edge length
  std::vector<double> dof_xyz;
  std::vector<int> en_ptr, en_dof;  // rows of P_e: node (cell, a) = sum en_w * dof
  std::vector<double> en_w;
  std::vector<double> ipx, ipy, ipz, ipw;
  std::vector<int> rowptr, colidx;
};

struct Oracle3 {
  int G = 0, S = 0;
  std::vector<Grid3> g;
  std::vector<double> mass, charge, nu;
  std::vector<int> sgrid;
  std::vector<long long> f_off, v_off;
  ld B[NQ][NB], dB[3][NQ][NB];  // basis values and reference gradients at the Gauss points
};

void build_tables(Oracle3* o) {
  ld v[3][3], d[3][3];
  for (int q = 0; q < 3; ++q) lagrange2(GX[q], v[q], d[q]);
  for (int q3 = 0; q3 < 3; ++q3)
    for (int q2 = 0; q2 < 3; ++q2)
      for (int q1 = 0; q1 < 3; ++q1)
        for (int a3 = 0; a3 < 3; ++a3)
          for (int a2 = 0; a2 < 3; ++a2)
            for (int a1 = 0; a1 < 3; ++a1) {
              const int q = q1 + 3 * q2 + 9 * q3, a = a1 + 3 * a2 + 9 * a3;
              o->B[q][a] = v[q1][a1] * v[q2][a2] * v[q3][a3];
              o->dB[0][q][a] = d[q1][a1] * v[q2][a2] * v[q3][a3];
              o->dB[1][q][a] = v[q1][a1] * d[q2][a2] * v[q3][a3];
              o->dB[2][q][a] = v[q1][a1] * v[q2][a2] * d[q3][a3];
            }
}

// O3: octree mesh, dofs, constraints.  Lattice coordinate of node a1 of cell (lev, i): X = (2 i + a1) << (L - lev),
// X in [0, 2 n 2^L]; the dof order is lexicographic in (Z, Y, X).
bool build_grid(Grid3* g) {
  const int L = g->levels, n = g->n;
  struct Leaf {
    int lev, i, j, k;
  };
  std::vector<Leaf> leaves;
  for (int k = 0; k < n; ++k)
    for (int j = 0; j < n; ++j)
      for (int i = 0; i < n; ++i) leaves.push_back(Leaf{0, i, j, k});
  for (int l = 1; l <= L; ++l) {
    // refine every level-(l-1) leaf whose closure contains the origin (centre of the box): "refinement about the origin"
    std::vector<Leaf> next;
    const long long centre2 = (long long)n << (l - 1);  // 2 x centre in level-(l-1) cell units = n 2^(l-1)
    for (const Leaf& c : leaves) {
      auto touches = [&](int i) { return 2LL * i <= centre2 && centre2 <= 2LL * (i + 1); };
      if (c.lev == l - 1 && touches(c.i) && touches(c.j) && touches(c.k)) {
        for (int dk = 0; dk < 2; ++dk)
          for (int dj = 0; dj < 2; ++dj)
            for (int di = 0; di < 2; ++di) next.push_back(Leaf{l, 2 * c.i + di, 2 * c.j + dj, 2 * c.k + dk});
      } else {
        next.push_back(c);
      }
    }
    leaves.swap(next);
  }
  g->n_cells = (int)leaves.size();
  const long long W = ((long long)2 * n << L) + 1;
  auto key = [&](long long X, long long Y, long long Z) { return (Z * W + Y) * W + X; };
  // all node lattice points
  std::map<long long, int> point_id;  // key -> index into pts
  struct Pt {
    long long X, Y, Z;
  };
  std::vector<Pt> pts;
  std::vector<int> cell_pt(g->n_cells * NB);
  for (int e = 0; e < g->n_cells; ++e) {
    const Leaf& c = leaves[e];
    const int sh = L - c.lev;
    for (int a3 = 0; a3 < 3; ++a3)
      for (int a2 = 0; a2 < 3; ++a2)
        for (int a1 = 0; a1 < 3; ++a1) {
          Pt p{(long long)(2 * c.i + a1) << sh, (long long)(2 * c.j + a2) << sh, (long long)(2 * c.k + a3) << sh};
          auto it = point_id.find(key(p.X, p.Y, p.Z));
          int id;
          if (it == point_id.end()) {
            id = (int)pts.size();
            point_id[key(p.X, p.Y, p.Z)] = id;
            pts.push_back(p);
          } else {
            id = it->second;
          }
          cell_pt[e * NB + a1 + 3 * a2 + 9 * a3] = id;
        }
  }
  // constraints: a point hangs if it lies in the closure of a leaf of which it is not a node; it then takes the value of
  // that leaf's Q2 interpolant (its trace on the face / edge the point lies on).  The coarsest such leaf is used.
  const int np = (int)pts.size();
  std::vector<std::vector<std::pair<int, ld>>> con(np);
  std::vector<char> hanging(np, 0);
  if (L > 0) {
    for (int p = 0; p < np; ++p) {
      int best = -1;
      for (int e = 0; e < g->n_cells; ++e) {
        const Leaf& c = leaves[e];
        const int sh = L - c.lev;
        const long long s = 1LL << sh, o[3] = {(long long)(2 * c.i) << sh, (long long)(2 * c.j) << sh, (long long)(2 * c.k) << sh};
        const long long P[3] = {pts[p].X, pts[p].Y, pts[p].Z};
        bool inside = true, is_node = true;
        for (int d = 0; d < 3; ++d) {
          if (P[d] < o[d] || P[d] > o[d] + 2 * s) inside = false;
          if ((P[d] - o[d]) % s != 0) is_node = false;
        }
        if (inside && !is_node && (best < 0 || leaves[e].lev < leaves[best].lev)) best = e;
      }
      if (best < 0) continue;
      hanging[p] = 1;
      const Leaf& c = leaves[best];
      const int sh = L - c.lev;
      const long long s = 1LL << sh;
      ld v[3][3], dd[3];
      const long long P[3] = {pts[p].X, pts[p].Y, pts[p].Z}, o[3] = {(long long)(2 * c.i) << sh, (long long)(2 * c.j) << sh, (long long)(2 * c.k) << sh};
      for (int d = 0; d < 3; ++d) lagrange2(-1 + (ld)(P[d] - o[d]) / (ld)s, v[d], dd);
      for (int a3 = 0; a3 < 3; ++a3)
        for (int a2 = 0; a2 < 3; ++a2)
          for (int a1 = 0; a1 < 3; ++a1) {
            const ld w = v[0][a1] * v[1][a2] * v[2][a3];
            if (w != 0) con[p].push_back(std::make_pair(cell_pt[best * NB + a1 + 3 * a2 + 9 * a3], w));
          }
    }
  }
  // free points -> dofs in (Z, Y, X) order
  std::vector<std::pair<long long, int>> order;
  for (int p = 0; p < np; ++p)
    if (!hanging[p]) order.push_back(std::make_pair(key(pts[p].X, pts[p].Y, pts[p].Z), p));
  std::sort(order.begin(), order.end());
  g->n_dof = (int)order.size();
  std::vector<int> dof_of(np, -1);
  const double unit = 2.0 * g->half / (double)((long long)2 * n << L);
  g->dof_xyz.resize(3 * (size_t)g->n_dof);
  for (int I = 0; I < g->n_dof; ++I) {
    const int p = order[I].second;
    dof_of[p] = I;
    g->dof_xyz[3 * I] = -g->half + unit * (double)pts[p].X;
    g->dof_xyz[3 * I + 1] = -g->half + unit * (double)pts[p].Y;
    g->dof_xyz[3 * I + 2] = -g->half + unit * (double)pts[p].Z;
  }
  // rows of P_e (constraint chains resolved by repeated substitution)
  g->en_ptr.assign(1, 0);
  for (int e = 0; e < g->n_cells; ++e)
    for (int a = 0; a < NB; ++a) {
      std::vector<std::pair<int, ld>> work(1, std::make_pair(cell_pt[e * NB + a], (ld)1)), nxt;
      for (int depth = 0; depth < 8; ++depth) {
        bool again = false;
        nxt.clear();
        for (auto& pw : work) {
          if (!hanging[pw.first]) {
            nxt.push_back(pw);
            continue;
          }
          again = true;
          for (auto& mw : con[pw.first]) nxt.push_back(std::make_pair(mw.first, pw.second * mw.second));
        }
        work.swap(nxt);
        if (!again) break;
        if (depth == 7) return false;
      }
      std::map<int, ld> merged;
      for (auto& pw : work) merged[dof_of[pw.first]] += pw.second;
      for (auto& dw : merged)
        if (dw.second != 0) {
          g->en_dof.push_back(dw.first);
          g->en_w.push_back((double)dw.second);
        }
      g->en_ptr.push_back((int)g->en_dof.size());
    }
  // O4: cells and integration points
  g->cx0.resize(g->n_cells);
  g->cy0.resize(g->n_cells);
  g->cz0.resize(g->n_cells);
  g->ch.resize(g->n_cells);
  g->n_ip = g->n_cells * NQ;
  g->ipx.resize(g->n_ip);
  g->ipy.resize(g->n_ip);
  g->ipz.resize(g->n_ip);
  g->ipw.resize(g->n_ip);
  for (int e = 0; e < g->n_cells; ++e) {
    const Leaf& c = leaves[e];
    const double h = 2.0 * g->half / (double)((long long)n << c.lev);
    g->ch[e] = h;
    g->cx0[e] = -g->half + c.i * h;
    g->cy0[e] = -g->half + c.j * h;
    g->cz0[e] = -g->half + c.k * h;
    for (int q3 = 0; q3 < 3; ++q3)
      for (int q2 = 0; q2 < 3; ++q2)
        for (int q1 = 0; q1 < 3; ++q1) {
          const int ip = e * NQ + q1 + 3 * q2 + 9 * q3;
          g->ipx[ip] = (double)(g->cx0[e] + 0.5L * h * (1 + GX[q1]));
          g->ipy[ip] = (double)(g->cy0[e] + 0.5L * h * (1 + GX[q2]));
          g->ipz[ip] = (double)(g->cz0[e] + 0.5L * h * (1 + GX[q3]));
          g->ipw[ip] = (double)(GW[q1] * GW[q2] * GW[q3] * 0.125L * h * h * h);
        }
  }
  // structural CSR pattern: every pair of dofs met in one cell
  std::vector<std::vector<int>> rows(g->n_dof);
  for (int e = 0; e < g->n_cells; ++e) {
    std::vector<int> touched(g->en_dof.begin() + g->en_ptr[e * NB], g->en_dof.begin() + g->en_ptr[(e + 1) * NB]);
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
  return true;
}

// O6: the Landau tensor.  out = (xx, xy, xz, yy, yz, zz); zero for coincident points (reading A2).
inline bool tensor3(const ld* v, const ld* vb, ld* U) {
  const ld u[3] = {v[0] - vb[0], v[1] - vb[1], v[2] - vb[2]};
  const ld u2 = u[0] * u[0] + u[1] * u[1] + u[2] * u[2];
  const ld scale = v[0] * v[0] + v[1] * v[1] + v[2] * v[2] + vb[0] * vb[0] + vb[1] * vb[1] + vb[2] * vb[2];
  if (u2 <= 1e-20L * scale) {
    for (int k = 0; k < 6; ++k) U[k] = 0;
    return false;
  }
  const ld inv3 = 1 / (u2 * sqrtl(u2));
  U[0] = (u2 - u[0] * u[0]) * inv3;
  U[1] = -u[0] * u[1] * inv3;
  U[2] = -u[0] * u[2] * inv3;
  U[3] = (u2 - u[1] * u[1]) * inv3;
  U[4] = -u[1] * u[2] * inv3;
  U[5] = (u2 - u[2] * u[2]) * inv3;
  return true;
}

// O5: f and its gradient at the integration points of species s (P_e applied to the nodal vector first)
void fields_at_ips(const Oracle3* o, int s, const double* f, std::vector<ld>* out /* [n_ip][4] */) {
  const Grid3& g = o->g[o->sgrid[s]];
  const double* fs = f + o->f_off[s];
  out->assign((size_t)g.n_ip * 4, 0);
  for (int e = 0; e < g.n_cells; ++e) {
    ld nodal[NB];
    for (int a = 0; a < NB; ++a) {
      ld v = 0;
      for (int p = g.en_ptr[e * NB + a]; p < g.en_ptr[e * NB + a + 1]; ++p) v += (ld)g.en_w[p] * fs[g.en_dof[p]];
      nodal[a] = v;
    }
    const ld sc = 2 / (ld)g.ch[e];
    for (int q = 0; q < NQ; ++q) {
      ld v = 0, gx = 0, gy = 0, gz = 0;
      for (int a = 0; a < NB; ++a) {
        v += o->B[q][a] * nodal[a];
        gx += o->dB[0][q][a] * nodal[a];
        gy += o->dB[1][q][a] * nodal[a];
        gz += o->dB[2][q][a] * nodal[a];
      }
      ld* dst = &(*out)[(size_t)(e * NQ + q) * 4];
      dst[0] = v;
      dst[1] = sc * gx;
      dst[2] = sc * gy;
      dst[3] = sc * gz;
    }
  }
}

// O7: inner integral at one field point for field species alpha: D (6) and K (3), all source species
void inner_point(const Oracle3* o, int alpha, const std::vector<std::vector<ld>>& fields, const ld* x, ld* DK) {
  for (int k = 0; k < 9; ++k) DK[k] = 0;
  const ld ma = o->mass[alpha];
  for (int beta = 0; beta < o->S; ++beta) {
    const Grid3& gb = o->g[o->sgrid[beta]];
    const std::vector<ld>& fb = fields[beta];
    ld GD[6] = {0, 0, 0, 0, 0, 0}, GK[3] = {0, 0, 0};
    for (int j = 0; j < gb.n_ip; ++j) {
      const ld xb[3] = {gb.ipx[j], gb.ipy[j], gb.ipz[j]};
      ld U[6];
      if (!tensor3(x, xb, U)) continue;
      const ld w = gb.ipw[j];
      const ld fj = w * fb[4 * (size_t)j], g0 = w * fb[4 * (size_t)j + 1], g1 = w * fb[4 * (size_t)j + 2], g2 = w * fb[4 * (size_t)j + 3];
      for (int k = 0; k < 6; ++k) GD[k] += U[k] * fj;
      GK[0] += U[0] * g0 + U[1] * g1 + U[2] * g2;
      GK[1] += U[1] * g0 + U[3] * g1 + U[4] * g2;
      GK[2] += U[2] * g0 + U[4] * g1 + U[5] * g2;
    }
    const ld nu = o->nu[alpha * o->S + beta], mb = o->mass[beta];
    for (int k = 0; k < 6; ++k) DK[k] += nu / (ma * ma) * GD[k];
    for (int k = 0; k < 3; ++k) DK[6 + k] += nu / (ma * mb) * GK[k];
  }
}

void inner_integral(const Oracle3* o, const double* f, std::vector<std::vector<ld>>* fields, std::vector<std::vector<ld>>* DK) {
  fields->resize(o->S);
  DK->resize(o->S);
  for (int s = 0; s < o->S; ++s) fields_at_ips(o, s, f, &(*fields)[s]);
  for (int a = 0; a < o->S; ++a) {
    const Grid3& g = o->g[o->sgrid[a]];
    (*DK)[a].assign((size_t)g.n_ip * 9, 0);
#pragma omp parallel for schedule(dynamic, 16)
    for (int i = 0; i < g.n_ip; ++i) {
      const ld x[3] = {g.ipx[i], g.ipy[i], g.ipz[i]};
      inner_point(o, a, *fields, x, &(*DK)[a][(size_t)i * 9]);
    }
  }
}

// symmetric D as a full 3 x 3
inline ld Dfull(const ld* d, int r, int c) {
  static const int idx[3][3] = {{0, 1, 2}, {1, 3, 4}, {2, 4, 5}};
  return d[idx[r][c]];
}

// O8 + O9: element matrices of M/dt - J and assembly through P_e^T . P_e into the CSR of the species' grid
void assemble_species(const Oracle3* o, int s, const std::vector<ld>& DK, ld inv_dt, bool mass_only, double* vals) {
  const Grid3& g = o->g[o->sgrid[s]];
  std::vector<ld> acc(g.nnz, 0);
  for (int e = 0; e < g.n_cells; ++e) {
    const ld sc = 2 / (ld)g.ch[e];
    std::vector<ld> A(NB * NB, 0);
    for (int q = 0; q < NQ; ++q) {
      const ld w = g.ipw[e * NQ + q];
      const ld* dk = mass_only ? nullptr : &DK[(size_t)(e * NQ + q) * 9];
      for (int a = 0; a < NB; ++a) {
        const ld ga[3] = {sc * o->dB[0][q][a], sc * o->dB[1][q][a], sc * o->dB[2][q][a]};
        for (int c = 0; c < NB; ++c) {
          ld v = inv_dt * o->B[q][a] * o->B[q][c];
          if (dk) {
            const ld gc[3] = {sc * o->dB[0][q][c], sc * o->dB[1][q][c], sc * o->dB[2][q][c]};
            ld dterm = 0, kterm = 0;
            for (int r = 0; r < 3; ++r) {
              for (int cc = 0; cc < 3; ++cc) dterm += ga[r] * Dfull(dk, r, cc) * gc[cc];
              kterm += ga[r] * dk[6 + r];
            }
            v += dterm - kterm * o->B[q][c];
          }
          A[a * NB + c] += w * v;
        }
      }
    }
    for (int a = 0; a < NB; ++a)
      for (int pa = g.en_ptr[e * NB + a]; pa < g.en_ptr[e * NB + a + 1]; ++pa) {
        const int I = g.en_dof[pa];
        const int* rb = &g.colidx[g.rowptr[I]];
        const int* re = &g.colidx[0] + g.rowptr[I + 1];
        for (int c = 0; c < NB; ++c)
          for (int pc = g.en_ptr[e * NB + c]; pc < g.en_ptr[e * NB + c + 1]; ++pc) {
            const int slot = (int)(std::lower_bound(rb, re, g.en_dof[pc]) - &g.colidx[0]);
            acc[slot] += (ld)g.en_w[pa] * (ld)g.en_w[pc] * A[a * NB + c];
          }
      }
  }
  for (int n = 0; n < g.nnz; ++n) vals[n] = (double)acc[n];
}

// O10: rhs = J[f] f, rhs_a = sum_q w_q [ -grad phi_a . D grad f + (grad phi_a . K) f ]
void apply_species(const Oracle3* o, int s, const std::vector<ld>& fld, const std::vector<ld>& DK, double* rhs) {
  const Grid3& g = o->g[o->sgrid[s]];
  std::vector<ld> acc(g.n_dof, 0);
  for (int e = 0; e < g.n_cells; ++e) {
    const ld sc = 2 / (ld)g.ch[e];
    ld r[NB];
    for (int a = 0; a < NB; ++a) r[a] = 0;
    for (int q = 0; q < NQ; ++q) {
      const size_t ip = (size_t)(e * NQ + q);
      const ld w = g.ipw[ip];
      const ld* dk = &DK[ip * 9];
      const ld* fq = &fld[ip * 4];
      ld flux[3];
      for (int rr = 0; rr < 3; ++rr) {
        ld v = 0;
        for (int cc = 0; cc < 3; ++cc) v += Dfull(dk, rr, cc) * fq[1 + cc];
        flux[rr] = -v + dk[6 + rr] * fq[0];
      }
      for (int a = 0; a < NB; ++a)
        r[a] += w * sc * (o->dB[0][q][a] * flux[0] + o->dB[1][q][a] * flux[1] + o->dB[2][q][a] * flux[2]);
    }
    for (int a = 0; a < NB; ++a)
      for (int pa = g.en_ptr[e * NB + a]; pa < g.en_ptr[e * NB + a + 1]; ++pa) acc[g.en_dof[pa]] += (ld)g.en_w[pa] * r[a];
  }
  for (int I = 0; I < g.n_dof; ++I) rhs[I] = (double)acc[I];
}

}  // namespace

extern "C" {

void* orc3_create(int n_grids, const double* half, const int* n, const int* levels, int n_species, const double* mass,
                  const double* charge, const int* grid, const double* nu) {
  Oracle3* o = new Oracle3();
  o->G = n_grids;
  o->S = n_species;
  build_tables(o);
  o->g.resize(n_grids);
  for (int g = 0; g < n_grids; ++g) {
    o->g[g].half = half[g];
    o->g[g].n = n[g];
    o->g[g].levels = levels[g];
    if (!build_grid(&o->g[g])) {
      delete o;
      return nullptr;
    }
  }
  long long fo = 0, vo = 0;
  for (int s = 0; s < n_species; ++s) {
    o->mass.push_back(mass[s]);
    o->charge.push_back(charge[s]);
    o->sgrid.push_back(grid[s]);
    o->f_off.push_back(fo);
    o->v_off.push_back(vo);
    fo += o->g[grid[s]].n_dof;
    vo += o->g[grid[s]].nnz;
  }
  o->f_off.push_back(fo);
  o->v_off.push_back(vo);
  o->nu.resize((size_t)n_species * n_species);
  for (int a = 0; a < n_species; ++a)
    for (int b = 0; b < n_species; ++b)
      o->nu[a * n_species + b] = nu ? nu[a * n_species + b] : charge[a] * charge[a] * charge[b] * charge[b];
  return o;
}
void orc3_destroy(void* h) { delete (Oracle3*)h; }
void orc3_sizes(void* h, int* n_dof, int* nnz, int* n_ip, int* n_cells) {
  Oracle3* o = (Oracle3*)h;
  for (int g = 0; g < o->G; ++g) {
    n_dof[g] = o->g[g].n_dof;
    nnz[g] = o->g[g].nnz;
    n_ip[g] = o->g[g].n_ip;
    n_cells[g] = o->g[g].n_cells;
  }
}
void orc3_dof_coords(void* h, int g, double* xyz) {
  Oracle3* o = (Oracle3*)h;
  memcpy(xyz, o->g[g].dof_xyz.data(), sizeof(double) * o->g[g].dof_xyz.size());
}
void orc3_pattern(void* h, int g, int* rowptr, int* colidx) {
  Oracle3* o = (Oracle3*)h;
  memcpy(rowptr, o->g[g].rowptr.data(), sizeof(int) * o->g[g].rowptr.size());
  memcpy(colidx, o->g[g].colidx.data(), sizeof(int) * o->g[g].colidx.size());
}
void orc3_ip_table(void* h, int g, double* x, double* y, double* z, double* w) {
  Oracle3* o = (Oracle3*)h;
  const Grid3& gr = o->g[g];
  memcpy(x, gr.ipx.data(), sizeof(double) * gr.n_ip);
  memcpy(y, gr.ipy.data(), sizeof(double) * gr.n_ip);
  memcpy(z, gr.ipz.data(), sizeof(double) * gr.n_ip);
  memcpy(w, gr.ipw.data(), sizeof(double) * gr.n_ip);
}
void orc3_tensor(const double* v, const double* vb, double* out6) {
  const ld a[3] = {v[0], v[1], v[2]}, b[3] = {vb[0], vb[1], vb[2]};
  ld U[6];
  tensor3(a, b, U);
  for (int k = 0; k < 6; ++k) out6[k] = (double)U[k];
}
// fields (f, grad f) of one species at its grid's integration points, [n_ip][4]
void orc3_fields(void* h, const double* f, int s, double* out) {
  Oracle3* o = (Oracle3*)h;
  std::vector<ld> fld;
  fields_at_ips(o, s, f, &fld);
  for (size_t k = 0; k < fld.size(); ++k) out[k] = (double)fld[k];
}
// D (xx, xy, xz, yy, yz, zz) and K (x, y, z) of every species at its integration points: out[species] -> [n_ip][9], concatenated
void orc3_inner(void* h, const double* f, double* out) {
  Oracle3* o = (Oracle3*)h;
  std::vector<std::vector<ld>> fields, DK;
  inner_integral(o, f, &fields, &DK);
  size_t off = 0;
  for (int s = 0; s < o->S; ++s) {
    for (size_t k = 0; k < DK[s].size(); ++k) out[off + k] = (double)DK[s][k];
    off += DK[s].size();
  }
}
// inner integral of field species alpha at arbitrary points, with the source fields GIVEN at the integration points
// (fsrc[beta] -> [n_ip(beta)][4]: f, grad f): for the closed-form pin with analytic sources
void orc3_inner_at_points(void* h, int alpha, const double* const* fsrc, const double* pts, int npts, double* out) {
  Oracle3* o = (Oracle3*)h;
  std::vector<std::vector<ld>> fields(o->S);
  for (int s = 0; s < o->S; ++s) {
    const int n = o->g[o->sgrid[s]].n_ip * 4;
    fields[s].resize(n);
    for (int k = 0; k < n; ++k) fields[s][k] = fsrc[s][k];
  }
  for (int p = 0; p < npts; ++p) {
    const ld x[3] = {pts[3 * p], pts[3 * p + 1], pts[3 * p + 2]};
    ld DK[9];
    inner_point(o, alpha, fields, x, DK);
    for (int k = 0; k < 9; ++k) out[9 * p + k] = (double)DK[k];
  }
}
void orc3_mass(void* h, int g, double* vals) {
  Oracle3* o = (Oracle3*)h;
  for (int s = 0; s < o->S; ++s)
    if (o->sgrid[s] == g) {
      std::vector<ld> none;
      assemble_species(o, s, none, 1, true, vals);
      return;
    }
}
void orc3_jacobian(void* h, const double* f, double dt, double* vals) {
  Oracle3* o = (Oracle3*)h;
  std::vector<std::vector<ld>> fields, DK;
  inner_integral(o, f, &fields, &DK);
  const ld inv_dt = std::isinf(dt) ? 0 : 1 / (ld)dt;
#pragma omp parallel for schedule(dynamic, 1)
  for (int s = 0; s < o->S; ++s) assemble_species(o, s, DK[s], inv_dt, false, vals + o->v_off[s]);
}
void orc3_apply(void* h, const double* f, double* rhs) {
  Oracle3* o = (Oracle3*)h;
  std::vector<std::vector<ld>> fields, DK;
  inner_integral(o, f, &fields, &DK);
  for (int s = 0; s < o->S; ++s) apply_species(o, s, fields[s], DK[s], rhs + o->f_off[s]);
}
int orc3_threads() {
#ifdef _OPENMP
  int n = 1;
#pragma omp parallel
  {
#pragma omp single
    n = omp_get_num_threads();
  }
  return n;
#else
  return 1;
#endif
}

}  // extern "C"
