// landau_oracle.cpp -- TEST INFRASTRUCTURE ONLY (oracle).
//
// Plain, slow, obviously-correct CPU restatement of the discrete 2V (axisymmetric r,z) Landau
// collision operator of arxiv 2209.03228 ("PAPER.md"), used only by tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs.  It shares no code, header, table or constant
// with the CUDA product path (paper_2209_03228_b200/csrc/) and the product never links or calls it.
//
// What it follows (PAPER.md line : passage):
//   * eq. (2.1), PAPER.md:44-48  -- C[fa,fb] = nu_ab (m0/ma) div INT U . ((m0/ma) fb grad fa - (m0/mb) fa grad fb)
//   * eq. (2.3), PAPER.md:59-64  -- D = sum_b INT U fb,  K = sum_b INT U . grad fb
//   * eq. (2.4), PAPER.md:68-71  -- weak form after integration by parts (sign reading A4 of DESIGN.md)
//   * PAPER.md:73                -- the sparse Jacobian freezes D(x), K(x) (inner integrals not linearised)
//   * PAPER.md:75-77             -- shifted matrix; we output M/dt - J (reading A15)
//   * PAPER.md:92 (sec. 2.3)     -- 2V cylindrical coordinates; the tensor is the azimuthal average of the
//                                   3-D Landau tensor (the paper only cites [12] App. A; derivation in DESIGN.md)
//   * PAPER.md:125               -- quadtree AMR grid with hanging nodes, no essential BCs (14 cells/142 eqs pin)
//   * PAPER.md:225-229 (sec. 5.2) -- unstructured grids of quadrilateral (tensor) cells: straight-sided cells, bilinear
//                                   reference map, gradient transformation J^-T per integration point (orc_create_meshes)
//
// Step by step, in the order of DESIGN.md "oracle steps" O1..O10.  No blocking, fusion or reordering:
// every batch entry recomputes every tensor.  Inner sums accumulate in long double; the tensor itself is
// evaluated in long double from cancellation-free AGM sums.  The only parallelism is an OpenMP
// "parallel for" over field points i (used for the timed CPU baseline).
//
// Parity pins (tests/test_oracle_*.py): P1 Gauss/Lagrange identities, P2 mass-matrix closed form,
// P3 tensor identities, P4 closed form vs brute-force azimuthal quadrature of the 3-D tensor and K,E vs
// std::comp_ellint, P5 Rosenbluth closed forms for a Maxwellian, P6 conservation to round-off,
// P7 equilibrium trend, P8 brute force on a tiny grid, P9 paper's mesh statistics (14/142/22.2),
// P10 / P11 the relaxation rates of PAPER.md Appendix B at t = 0 (bi-Maxwellian isotropisation rate nu_T, two-species
// thermal equilibration rate nu_bar) from the moments of the applied operator: they fix nu_ab, t0 and the weights.
// Unpinned: temperature HISTORIES over many collision times (Fig. 5 of the paper: needs its time integrator).

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <string>
#include <utility>
#include <vector>

typedef long double ld;

namespace {

const ld PI_L = 3.14159265358979323846264338327950288419716939937510L;

// ---------------------------------------------------------------------------------------------
// O1  Gauss-Legendre nodes/weights on [-1,1]: Newton iteration on P_n (PAPER.md:309-313 fixes
//     (k+1)^2 points per Qk cell).
// ---------------------------------------------------------------------------------------------
void gauss_legendre(int n, ld* x, ld* w) {
  for (int i = 0; i < n; i++) {
    ld t = cosl(PI_L * (i + 0.75L) / (n + 0.5L));
    ld dp = 0;
    for (int it = 0; it < 100; it++) {
      ld p0 = 1, p1 = t;
      for (int l = 2; l <= n; l++) {
        ld p2 = ((2 * l - 1) * t * p1 - (l - 1) * p0) / l;
        p0 = p1;
        p1 = p2;
      }
      if (n == 0) p1 = 1;
      dp = n * (t * p1 - p0) / (t * t - 1);
      ld dt = p1 / dp;
      t -= dt;
      if (fabsl(dt) < 1e-19L) break;
    }
    // re-evaluate derivative at the converged root
    ld p0 = 1, p1 = t;
    for (int l = 2; l <= n; l++) {
      ld p2 = ((2 * l - 1) * t * p1 - (l - 1) * p0) / l;
      p0 = p1;
      p1 = p2;
    }
    dp = n * (t * p1 - p0) / (t * t - 1);
    x[n - 1 - i] = t;  // ascending
    w[n - 1 - i] = 2 / ((1 - t * t) * dp * dp);
  }
}

// ---------------------------------------------------------------------------------------------
// O2  1-D Lagrange basis of degree k on k+1 EQUISPACED nodes of [-1,1] (reading A9).
// ---------------------------------------------------------------------------------------------
void lagrange_1d(int k, ld xi, ld* val, ld* der) {
  std::vector<ld> nodes(k + 1);
  for (int c = 0; c <= k; c++) nodes[c] = -1 + 2 * (ld)c / k;
  for (int c = 0; c <= k; c++) {
    ld v = 1;
    for (int d = 0; d <= k; d++)
      if (d != c) v *= (xi - nodes[d]) / (nodes[c] - nodes[d]);
    val[c] = v;
    ld s = 0;
    for (int e = 0; e <= k; e++) {
      if (e == c) continue;
      ld t = 1 / (nodes[c] - nodes[e]);
      for (int d = 0; d <= k; d++)
        if (d != c && d != e) t *= (xi - nodes[d]) / (nodes[c] - nodes[d]);
      s += t;
    }
    der[c] = s;
  }
}

// ---------------------------------------------------------------------------------------------
// O6  Complete elliptic pieces by the arithmetic-geometric mean, all sums of positive terms.
//     With Delta = sqrt(1 - m sin^2 t), all integrals over t in [0, pi/2]:
//        K  = INT 1/Delta            E  = INT Delta
//        P0 = INT Delta^-3           = E/m'
//        Dc = INT cos^2 Delta^-3     = (K-E)/m
//        P1 = INT sin^2 Delta^-3     = P0 - Dc
//        Q  = INT sin^2 cos^2 Delta^-3 = ((2-m)K - 2E)/m^2
//        P2 = INT sin^4 Delta^-3     = P1 - Q
//     AGM: a0=1, b0=sqrt(m'), c0^2=m; a_{n+1}=(a_n+b_n)/2, b_{n+1}=sqrt(a_n b_n), c_{n+1}=(a_n-b_n)/2.
//        K = pi/(2 a_inf),  K-E = K sum_{n>=0} 2^{n-1} c_n^2      (textbook, e.g. Abramowitz-Stegun 17.6)
//     Writing d_n = c_n/m (d_1 = 1/(2(1+sqrt m')), d_{n+1} = m d_n^2/(4 a_{n+1}) from a_{n+1}c_{n+1}=c_n^2/4)
//     and T = sum_{n>=1} 2^{n-1} d_n^2:   K-E = K (m/2 + m^2 T), hence
//        Dc = K (1/2 + m T),   Q = 2 K T,   E = K (1 - m/2 - m^2 T)
//     -- no subtraction of nearly equal numbers for any m in (0,1) except the mild one in E as m->1.
//     m' is passed in separately (computed from the geometry as s-/s+, never as 1-m).
// ---------------------------------------------------------------------------------------------
struct Ellip {
  ld K, E, P0, P1, Dc, Q, P2;
};

Ellip ellip_agm(ld m, ld mp) {
  ld a = 1, b = sqrtl(mp);
  ld d = 1 / (2 * (1 + b));  // d_1
  ld T = 0, pw = 1;          // pw = 2^{n-1}
  for (int n = 1; n < 64; n++) {
    ld an = (a + b) / 2;
    ld bn = sqrtl(a * b);
    // here (an, bn) = (a_n, b_n) and d = d_n
    T += pw * d * d;
    a = an;
    b = bn;
    if (pw * d * d < 1e-24L * T && fabsl(a - b) < 1e-19L * a) break;
    // d_{n+1} = m d_n^2 / (4 a_{n+1}),  a_{n+1} = (a_n+b_n)/2
    d = m * d * d / (4 * ((a + b) / 2));
    pw *= 2;
  }
  Ellip e;
  e.K = PI_L / (2 * a);
  e.Dc = e.K * (0.5L + m * T);
  e.Q = 2 * e.K * T;
  e.E = e.K * (1 - m / 2 - m * m * T);
  e.P0 = e.E / mp;
  e.P1 = e.P0 - e.Dc;
  e.P2 = e.P1 - e.Q;
  return e;
}

// ---------------------------------------------------------------------------------------------
// O6  2V Landau tensor: azimuthal average of U(v,vb) = (|u|^2 I - u u^T)/|u|^3, u = v - vb,
//     v = (r,0,z), vb = (rb cos p, rb sin p, zb), e_r=(1,0,0), eb_r=(cos p, sin p, 0), e_z=eb_z=(0,0,1):
//        UD_ab = INT_0^2pi e_a.U.e_b dp   (contracts with grad f at the field point)
//        UK_ab = INT_0^2pi e_a.U.eb_b dp  (contracts with grad fb at the source point)
//     With p = pi - 2t: |u|^2 = s+ (1 - m sin^2 t), s+- = (r +- rb)^2 + dz^2, m = 4 r rb/s+, m' = s-/s+,
//     c = 4/s+^{3/2}:
//        UD_rr = c (4 rb^2 Q + dz^2 P0)            UK_rr = c (4 r rb Q + dz^2 m P2)
//        UD_zz = c ((r-rb)^2 P0 + 4 r rb Dc)       UK_zz = UD_zz
//        UD_rz = -dz c ((r-rb) P0 + 2 rb Dc)       UK_rz = UD_rz
//                                                  UK_zr =  dz c ((rb-r) P0 + 2 r Dc)
//     (derivation in DESIGN.md; pinned against tensor_quadrature below, test P4).
//     Coincident points (s- <= 1e-20 s+): contribution defined as zero (reading A2); returns false.
// ---------------------------------------------------------------------------------------------
struct Tensor2V {
  ld UDrr, UDrz, UDzz, UKrr, UKzr;
};

bool tensor_closed(ld r, ld z, ld rb, ld zb, Tensor2V* t) {
  ld dz = z - zb;
  ld sp = (r + rb) * (r + rb) + dz * dz;
  ld sm = (r - rb) * (r - rb) + dz * dz;
  if (sm <= 1e-20L * sp) {
    t->UDrr = t->UDrz = t->UDzz = t->UKrr = t->UKzr = 0;
    return false;
  }
  ld m = 4 * r * rb / sp;
  ld mp = sm / sp;
  Ellip e = ellip_agm(m, mp);
  ld c = 4 / (sp * sqrtl(sp));
  t->UDrr = c * (4 * rb * rb * e.Q + dz * dz * e.P0);
  t->UDzz = c * ((r - rb) * (r - rb) * e.P0 + 4 * r * rb * e.Dc);
  t->UDrz = -dz * c * ((r - rb) * e.P0 + 2 * rb * e.Dc);
  t->UKrr = c * (4 * r * rb * e.Q + dz * dz * m * e.P2);
  t->UKzr = dz * c * ((rb - r) * e.P0 + 2 * r * e.Dc);
  return true;
}

// The plain definition: periodic trapezoid rule in the azimuth on the 3-D tensor.  Test mode only.
// out = {UDrr, UDrz, UDzz, UKrr, UKrz, UKzr, UKzz, UDzr}
void tensor_quadrature(ld r, ld z, ld rb, ld zb, int nphi, ld* out) {
  for (int k = 0; k < 8; k++) out[k] = 0;
  for (int p = 0; p < nphi; p++) {
    ld phi = 2 * PI_L * (p + 0.5L) / nphi;
    ld cp = cosl(phi), sn = sinl(phi);
    ld u[3] = {r - rb * cp, -rb * sn, z - zb};
    ld u2 = u[0] * u[0] + u[1] * u[1] + u[2] * u[2];
    ld u3 = u2 * sqrtl(u2);
    ld U[3][3];
    for (int a = 0; a < 3; a++)
      for (int b = 0; b < 3; b++) U[a][b] = ((a == b ? u2 : 0) - u[a] * u[b]) / u3;
    ld er[3] = {1, 0, 0}, ez[3] = {0, 0, 1}, ebr[3] = {cp, sn, 0};
    ld* ea[2] = {er, ez};
    ld* ebD[2] = {er, ez};
    ld* ebK[2] = {ebr, ez};
    ld UD[2][2], UK[2][2];
    for (int a = 0; a < 2; a++)
      for (int b = 0; b < 2; b++) {
        ld sD = 0, sK = 0;
        for (int x = 0; x < 3; x++)
          for (int y = 0; y < 3; y++) {
            sD += ea[a][x] * U[x][y] * ebD[b][y];
            sK += ea[a][x] * U[x][y] * ebK[b][y];
          }
        UD[a][b] = sD;
        UK[a][b] = sK;
      }
    out[0] += UD[0][0];
    out[1] += UD[0][1];
    out[2] += UD[1][1];
    out[3] += UK[0][0];
    out[4] += UK[0][1];
    out[5] += UK[1][0];
    out[6] += UK[1][1];
    out[7] += UD[1][0];
  }
  for (int k = 0; k < 8; k++) out[k] *= 2 * PI_L / nphi;
}

// ---------------------------------------------------------------------------------------------
// O3  Mesh, dofs, hanging-node constraints.
//     Integer lattice: one unit = base cell side / (k 2^L).  A level-l cell has side k 2^{L-l} units and
//     node spacing 2^{L-l}.  Quadtree rule (reading A12): for l = 1..L refine every level-(l-1) cell lying
//     inside the box [0, R/2^l] x [Zc - Zh/2^l, Zc + Zh/2^l]  (R = r extent, Zc = z centre, Zh = z half-extent).
// ---------------------------------------------------------------------------------------------
struct GridDesc {
  int kind;  // 0 uniform, 1 quadtree
  double r_max, z_min, z_max;
  int nr, nz, levels;
};
struct SpeciesDesc {
  double mass, charge;
  int grid;
};

struct Cell {
  long ix, iz;  // lattice origin
  int level;
};

struct Grid {
  GridDesc desc;
  int k, L;
  std::vector<Cell> cells;
  ld ur, uz;  // physical size of a lattice unit
  int n_dof;
  std::vector<long> dof_ix, dof_iz;
  // cell -> local node a -> list of (dof, weight)   (the rows of P_e)
  std::vector<std::vector<std::vector<std::pair<int, ld>>>> P;
  std::vector<int> rowptr, colidx;
  // integration points, cell-major: ip = cell*nq + q
  std::vector<ld> ip_r, ip_z, ip_w;
  // unstructured straight-sided quadrilaterals (sec. 5.2): the reference-to-physical map is bilinear, so
  // the gradient transformation differs from point to point.  gm[ip] = J^-T, (d/dr, d/dz) = gm (d/dxi, d/deta);
  // rectangular grids keep the two scale factors 2/hr, 2/hz of their cell.
  bool unstructured = false;
  std::vector<ld> gm;            // [ip][4]: m00 m01 m10 m11
  std::vector<ld> node_r, node_z;  // dof coordinates (unstructured grids)
  int n_ip() const { return (int)ip_r.size(); }
};

typedef std::pair<long, long> Key;
typedef std::vector<std::pair<Key, ld>> Combo;  // linear combination of lattice nodes

void build_mesh(Grid& g) {
  const int k = g.k;
  const GridDesc& d = g.desc;
  g.L = d.kind == 1 ? d.levels : 0;
  const int L = g.L;
  const long side0 = (long)k << L;
  g.ur = (ld)d.r_max / (d.nr * side0);
  g.uz = ((ld)d.z_max - (ld)d.z_min) / (d.nz * side0);
  std::vector<Cell> cur;
  for (int cz = 0; cz < d.nz; cz++)
    for (int cr = 0; cr < d.nr; cr++) cur.push_back(Cell{cr * side0, cz * side0, 0});
  const long R = d.nr * side0, Z = d.nz * side0;
  for (int l = 1; l <= L; l++) {
    // box in doubled lattice units to stay integral: r in [0, 2R/2^l], z in [Z - Z/2^l, Z + Z/2^l]
    long rhi2 = (2 * R) >> l, zlo2 = Z - (Z >> l), zhi2 = Z + (Z >> l);
    std::vector<Cell> nxt;
    for (const Cell& c : cur) {
      long side = (long)k << (L - c.level);
      bool inside = c.level == l - 1 && 2 * (c.ix + side) <= rhi2 && 2 * c.iz >= zlo2 && 2 * (c.iz + side) <= zhi2;
      if (!inside) {
        nxt.push_back(c);
        continue;
      }
      long h = side / 2;
      for (int bz = 0; bz < 2; bz++)
        for (int br = 0; br < 2; br++) nxt.push_back(Cell{c.ix + br * h, c.iz + bz * h, c.level + 1});
    }
    cur.swap(nxt);
  }
  g.cells = cur;

  // all lattice nodes touched by some cell
  std::map<Key, int> nodes;
  for (const Cell& c : g.cells) {
    long s = 1L << (L - c.level);
    for (int a2 = 0; a2 <= k; a2++)
      for (int a1 = 0; a1 <= k; a1++) nodes[Key(c.ix + a1 * s, c.iz + a2 * s)] = 0;
  }
  // hanging nodes: a node on an edge of a cell that is not one of that cell's own nodes is constrained to
  // the edge's k+1 nodes with the edge's Lagrange weights.
  std::map<Key, Combo> constraint;
  for (const Cell& c : g.cells) {
    long s = 1L << (L - c.level), side = k * s;
    for (const auto& nd : nodes) {
      long x = nd.first.first, z = nd.first.second;
      if (constraint.count(nd.first)) continue;
      for (int edge = 0; edge < 4; edge++) {
        // edges: 0 z=iz, 1 z=iz+side (along r); 2 r=ix, 3 r=ix+side (along z)
        bool along_r = edge < 2;
        long fixed = along_r ? (edge == 0 ? c.iz : c.iz + side) : (edge == 2 ? c.ix : c.ix + side);
        long pos = along_r ? x - c.ix : z - c.iz;
        long oth = along_r ? z : x;
        if (oth != fixed || pos < 0 || pos > side) continue;
        if (pos % s == 0) continue;  // one of the cell's own nodes
        std::vector<ld> val(k + 1), der(k + 1);
        lagrange_1d(k, -1 + 2 * (ld)pos / side, val.data(), der.data());
        Combo cb;
        for (int cidx = 0; cidx <= k; cidx++) {
          Key master = along_r ? Key(c.ix + cidx * s, fixed) : Key(fixed, c.iz + cidx * s);
          cb.push_back(std::make_pair(master, val[cidx]));
        }
        constraint[nd.first] = cb;
        break;
      }
    }
  }
  // dofs = unconstrained nodes, ordered by (z, r)  (reading A17: lexicographic, z-major)
  std::vector<Key> free_nodes;
  for (const auto& nd : nodes)
    if (!constraint.count(nd.first)) free_nodes.push_back(nd.first);
  std::sort(free_nodes.begin(), free_nodes.end(), [](const Key& a, const Key& b) {
    return a.second != b.second ? a.second < b.second : a.first < b.first;
  });
  std::map<Key, int> dof_of;
  g.n_dof = (int)free_nodes.size();
  g.dof_ix.resize(g.n_dof);
  g.dof_iz.resize(g.n_dof);
  for (int i = 0; i < g.n_dof; i++) {
    dof_of[free_nodes[i]] = i;
    g.dof_ix[i] = free_nodes[i].first;
    g.dof_iz[i] = free_nodes[i].second;
  }
  // resolve a node to free dofs (follows chains, although reading A12's meshes have none)
  struct Resolver {
    const std::map<Key, Combo>& con;
    const std::map<Key, int>& dof_of;
    void run(const Key& key, ld wgt, std::map<int, ld>& out, int depth) const {
      auto it = con.find(key);
      if (it == con.end()) {
        out[dof_of.at(key)] += wgt;
        return;
      }
      if (depth > 8) {
        fprintf(stderr, "oracle: constraint chain too deep\n");
        abort();
      }
      for (const auto& mw : it->second) run(mw.first, wgt * mw.second, out, depth + 1);
    }
  } resolver{constraint, dof_of};
  g.P.resize(g.cells.size());
  for (size_t e = 0; e < g.cells.size(); e++) {
    const Cell& c = g.cells[e];
    long s = 1L << (L - c.level);
    g.P[e].resize((k + 1) * (k + 1));
    for (int a2 = 0; a2 <= k; a2++)
      for (int a1 = 0; a1 <= k; a1++) {
        std::map<int, ld> out;
        resolver.run(Key(c.ix + a1 * s, c.iz + a2 * s), 1, out, 0);
        for (const auto& dw : out)
          if (dw.second != 0) g.P[e][a1 + (k + 1) * a2].push_back(dw);
      }
  }
  // structural CSR pattern: every pair of dofs reached from one cell
  std::vector<std::vector<int>> rows(g.n_dof);
  for (size_t e = 0; e < g.cells.size(); e++) {
    std::vector<int> touched;
    for (const auto& row : g.P[e])
      for (const auto& dw : row) touched.push_back(dw.first);
    std::sort(touched.begin(), touched.end());
    touched.erase(std::unique(touched.begin(), touched.end()), touched.end());
    for (int I : touched)
      for (int J : touched) rows[I].push_back(J);
  }
  g.rowptr.assign(g.n_dof + 1, 0);
  g.colidx.clear();
  for (int I = 0; I < g.n_dof; I++) {
    std::sort(rows[I].begin(), rows[I].end());
    rows[I].erase(std::unique(rows[I].begin(), rows[I].end()), rows[I].end());
    g.rowptr[I + 1] = g.rowptr[I] + (int)rows[I].size();
    g.colidx.insert(g.colidx.end(), rows[I].begin(), rows[I].end());
  }
}

struct Problem {
  int k, nq1, nb, nq;
  std::vector<Grid> grids;
  std::vector<SpeciesDesc> species;
  std::vector<ld> nu;  // S x S
  std::vector<ld> gx, gw;
  bool simplex = false;            // triangles: reference quadrature points / weights below, nodes (i/k, j/k)
  std::vector<ld> sx, se, sw;
  // basis tabulation at the Gauss points of the reference cell:
  // B[q][a], dBxi[q][a], dBeta[q][a]; q = q1 + nq1*q2, a = a1 + (k+1)*a2
  std::vector<ld> B, dBxi, dBeta;
  std::vector<long long> f_off;  // offset of species alpha inside one batch entry of f
  long long f_stride;
  std::vector<long long> v_off;  // offset of species alpha inside one batch entry of CSR values
  long long v_stride;
  int threads;
};

// O4  integration-point table: r = r0 + hr(1+xi)/2, z likewise, w = gw gw (hr hz/4) r.
void build_ips(const Problem& pb, Grid& g) {
  const int k = pb.k;
  g.ip_r.clear();
  g.ip_z.clear();
  g.ip_w.clear();
  for (const Cell& c : g.cells) {
    long s = 1L << (g.L - c.level);
    ld r0 = c.ix * g.ur, z0 = (ld)g.desc.z_min + c.iz * g.uz;
    ld hr = k * s * g.ur, hz = k * s * g.uz;
    for (int q2 = 0; q2 < pb.nq1; q2++)
      for (int q1 = 0; q1 < pb.nq1; q1++) {
        ld r = r0 + hr * (1 + pb.gx[q1]) / 2;
        ld z = z0 + hz * (1 + pb.gx[q2]) / 2;
        g.ip_r.push_back(r);
        g.ip_z.push_back(z);
        g.ip_w.push_back(pb.gw[q1] * pb.gw[q2] * (hr * hz / 4) * r);
      }
  }
}

void cell_sizes(const Grid& g, int e, ld* hr, ld* hz) {
  long s = 1L << (g.L - g.cells[e].level);
  *hr = g.k * s * g.ur;
  *hz = g.k * s * g.uz;
}

// physical gradient of a function with reference gradient (dxi, deta) at integration point q of cell e
inline void grad_phys(const Grid& g, int e, int ip, ld dxi, ld deta, ld* pr, ld* pz) {
  if (g.unstructured) {
    const ld* m = &g.gm[4 * (size_t)ip];
    *pr = m[0] * dxi + m[1] * deta;
    *pz = m[2] * dxi + m[3] * deta;
  } else {
    ld hr, hz;
    cell_sizes(g, e, &hr, &hz);
    *pr = (2 / hr) * dxi;
    *pz = (2 / hz) * deta;
  }
}

// O3'' + O4'' the same for triangles: affine map x = v0 + (v1 - v0) xi + (v2 - v0) eta, constant J per cell.
bool build_unstructured_simplex(const Problem& pb, Grid& g, int nv, const double* verts, int nc, const int* cells) {
  const int k = pb.k, nb = pb.nb;
  g.unstructured = true;
  g.L = 0;
  g.cells.assign(nc, Cell{0, 0, 0});
  ld scale = 0;
  for (int v = 0; v < 2 * nv; v++) scale = std::max(scale, fabsl((ld)verts[v]));
  const ld quantum = scale / (ld)(1L << 30);
  auto vr = [&](int e, int c) { return (ld)verts[2 * cells[3 * e + c]]; };
  auto vz = [&](int e, int c) { return (ld)verts[2 * cells[3 * e + c] + 1]; };
  std::map<Key, int> node_id;
  std::vector<Key> keys;
  std::vector<ld> nr, nz;
  std::vector<int> cell_node((size_t)nc * nb);
  for (int e = 0; e < nc; e++) {
    int a = 0;
    for (int j = 0; j <= k; j++)
      for (int i = 0; i <= k - j; i++, a++) {
        const ld xi = (ld)i / k, eta = (ld)j / k;
        const ld r = vr(e, 0) + (vr(e, 1) - vr(e, 0)) * xi + (vr(e, 2) - vr(e, 0)) * eta;
        const ld z = vz(e, 0) + (vz(e, 1) - vz(e, 0)) * xi + (vz(e, 2) - vz(e, 0)) * eta;
        const Key key((long)llroundl(z / quantum), (long)llroundl(r / quantum));
        auto it = node_id.find(key);
        int id;
        if (it == node_id.end()) {
          id = (int)keys.size();
          node_id[key] = id;
          keys.push_back(key);
          nr.push_back(r);
          nz.push_back(z);
        } else {
          id = it->second;
        }
        cell_node[(size_t)e * nb + a] = id;
      }
  }
  std::vector<int> order(keys.size());
  for (size_t i = 0; i < order.size(); i++) order[i] = (int)i;
  std::sort(order.begin(), order.end(), [&](int a, int b) { return keys[a] < keys[b]; });
  std::vector<int> dof_of(keys.size());
  g.n_dof = (int)keys.size();
  g.node_r.resize(g.n_dof);
  g.node_z.resize(g.n_dof);
  for (int I = 0; I < g.n_dof; I++) {
    dof_of[order[I]] = I;
    g.node_r[I] = nr[order[I]];
    g.node_z[I] = nz[order[I]];
  }
  g.P.assign(nc, std::vector<std::vector<std::pair<int, ld>>>(nb));
  for (int e = 0; e < nc; e++)
    for (int a = 0; a < nb; a++) g.P[e][a].push_back(std::make_pair(dof_of[cell_node[(size_t)e * nb + a]], (ld)1));
  std::vector<std::vector<int>> rows(g.n_dof);
  for (int e = 0; e < nc; e++) {
    std::vector<int> touched;
    for (const auto& row : g.P[e])
      for (const auto& dw : row) touched.push_back(dw.first);
    std::sort(touched.begin(), touched.end());
    touched.erase(std::unique(touched.begin(), touched.end()), touched.end());
    for (int I : touched)
      for (int J : touched) rows[I].push_back(J);
  }
  g.rowptr.assign(g.n_dof + 1, 0);
  g.colidx.clear();
  for (int I = 0; I < g.n_dof; I++) {
    std::sort(rows[I].begin(), rows[I].end());
    rows[I].erase(std::unique(rows[I].begin(), rows[I].end()), rows[I].end());
    g.rowptr[I + 1] = g.rowptr[I] + (int)rows[I].size();
    g.colidx.insert(g.colidx.end(), rows[I].begin(), rows[I].end());
  }
  for (int e = 0; e < nc; e++) {
    const ld J[4] = {vr(e, 1) - vr(e, 0), vr(e, 2) - vr(e, 0), vz(e, 1) - vz(e, 0), vz(e, 2) - vz(e, 0)};
    const ld det = J[0] * J[3] - J[1] * J[2];
    if (!(det > 0)) return false;
    for (int q = 0; q < pb.nq; q++) {
      const ld r = vr(e, 0) + J[0] * pb.sx[q] + J[1] * pb.se[q], z = vz(e, 0) + J[2] * pb.sx[q] + J[3] * pb.se[q];
      g.ip_r.push_back(r);
      g.ip_z.push_back(z);
      g.ip_w.push_back(pb.sw[q] * det * r);
      g.gm.push_back(J[3] / det);
      g.gm.push_back(-J[2] / det);
      g.gm.push_back(-J[1] / det);
      g.gm.push_back(J[0] / det);
    }
  }
  return true;
}

// O3' + O4' unstructured conforming mesh of straight-sided quadrilaterals (vertices (r, z), cells = 4 vertex ids,
// counter-clockwise).  Qk nodes sit at the images of the equispaced reference nodes under the cell's bilinear map; nodes
// of neighbouring cells that coincide are one dof (found geometrically: equal coordinates on a grid of 2^-30 of the mesh
// extent); dofs are ordered by (z, r) on that grid; no constraints.  Integration points: the images of the Gauss points,
// w = gw gw det(J) r with J the Jacobian of the bilinear map at the point.
bool build_unstructured(const Problem& pb, Grid& g, int nv, const double* verts, int nc, const int* cells) {
  if (pb.simplex) return build_unstructured_simplex(pb, g, nv, verts, nc, cells);
  const int k = pb.k, n1 = k + 1;
  g.unstructured = true;
  g.L = 0;
  g.cells.assign(nc, Cell{0, 0, 0});
  ld scale = 0;
  for (int v = 0; v < 2 * nv; v++) scale = std::max(scale, fabsl((ld)verts[v]));
  const ld quantum = scale / (ld)(1L << 30);
  auto bilinear = [&](int e, ld xi, ld eta, ld* r, ld* z, ld* J) {
    const ld N[4] = {(1 - xi) * (1 - eta) / 4, (1 + xi) * (1 - eta) / 4, (1 + xi) * (1 + eta) / 4, (1 - xi) * (1 + eta) / 4};
    const ld Nx[4] = {-(1 - eta) / 4, (1 - eta) / 4, (1 + eta) / 4, -(1 + eta) / 4};
    const ld Ne[4] = {-(1 - xi) / 4, -(1 + xi) / 4, (1 + xi) / 4, (1 - xi) / 4};
    *r = *z = 0;
    if (J) J[0] = J[1] = J[2] = J[3] = 0;
    for (int v = 0; v < 4; v++) {
      const ld vr = verts[2 * cells[4 * e + v]], vz = verts[2 * cells[4 * e + v] + 1];
      *r += N[v] * vr;
      *z += N[v] * vz;
      if (J) {
        J[0] += Nx[v] * vr;  // dr/dxi
        J[1] += Ne[v] * vr;  // dr/deta
        J[2] += Nx[v] * vz;  // dz/dxi
        J[3] += Ne[v] * vz;  // dz/deta
      }
    }
  };
  std::map<Key, int> node_id;  // (quantised z, quantised r) -> provisional id
  std::vector<Key> keys;
  std::vector<ld> nr, nz;
  std::vector<int> cell_node((size_t)nc * n1 * n1);
  for (int e = 0; e < nc; e++)
    for (int a2 = 0; a2 <= k; a2++)
      for (int a1 = 0; a1 <= k; a1++) {
        ld r, z;
        bilinear(e, -1 + 2 * (ld)a1 / k, -1 + 2 * (ld)a2 / k, &r, &z, nullptr);
        const Key key((long)llroundl(z / quantum), (long)llroundl(r / quantum));
        auto it = node_id.find(key);
        int id;
        if (it == node_id.end()) {
          id = (int)keys.size();
          node_id[key] = id;
          keys.push_back(key);
          nr.push_back(r);
          nz.push_back(z);
        } else {
          id = it->second;
        }
        cell_node[((size_t)e * n1 + a2) * n1 + a1] = id;
      }
  std::vector<int> order(keys.size());
  for (size_t i = 0; i < order.size(); i++) order[i] = (int)i;
  std::sort(order.begin(), order.end(), [&](int a, int b) { return keys[a] < keys[b]; });
  std::vector<int> dof_of(keys.size());
  g.n_dof = (int)keys.size();
  g.node_r.resize(g.n_dof);
  g.node_z.resize(g.n_dof);
  for (int I = 0; I < g.n_dof; I++) {
    dof_of[order[I]] = I;
    g.node_r[I] = nr[order[I]];
    g.node_z[I] = nz[order[I]];
  }
  g.P.assign(nc, std::vector<std::vector<std::pair<int, ld>>>(n1 * n1));
  for (int e = 0; e < nc; e++)
    for (int a = 0; a < n1 * n1; a++) g.P[e][a].push_back(std::make_pair(dof_of[cell_node[(size_t)e * n1 * n1 + a]], (ld)1));
  std::vector<std::vector<int>> rows(g.n_dof);
  for (int e = 0; e < nc; e++) {
    std::vector<int> touched;
    for (const auto& row : g.P[e])
      for (const auto& dw : row) touched.push_back(dw.first);
    std::sort(touched.begin(), touched.end());
    touched.erase(std::unique(touched.begin(), touched.end()), touched.end());
    for (int I : touched)
      for (int J : touched) rows[I].push_back(J);
  }
  g.rowptr.assign(g.n_dof + 1, 0);
  g.colidx.clear();
  for (int I = 0; I < g.n_dof; I++) {
    std::sort(rows[I].begin(), rows[I].end());
    rows[I].erase(std::unique(rows[I].begin(), rows[I].end()), rows[I].end());
    g.rowptr[I + 1] = g.rowptr[I] + (int)rows[I].size();
    g.colidx.insert(g.colidx.end(), rows[I].begin(), rows[I].end());
  }
  for (int e = 0; e < nc; e++)
    for (int q2 = 0; q2 < pb.nq1; q2++)
      for (int q1 = 0; q1 < pb.nq1; q1++) {
        ld r, z, J[4];
        bilinear(e, pb.gx[q1], pb.gx[q2], &r, &z, J);
        const ld det = J[0] * J[3] - J[1] * J[2];
        if (!(det > 0)) return false;  // inverted or clockwise cell
        g.ip_r.push_back(r);
        g.ip_z.push_back(z);
        g.ip_w.push_back(pb.gw[q1] * pb.gw[q2] * det * r);
        // J^-1 = 1/det [ dz/deta, -dr/deta ; -dz/dxi, dr/dxi ] (rows: xi_r xi_z ; eta_r eta_z); gm = J^-T
        g.gm.push_back(J[3] / det);
        g.gm.push_back(-J[2] / det);
        g.gm.push_back(-J[1] / det);
        g.gm.push_back(J[0] / det);
      }
  return true;
}

// ---------------------------------------------------------------------------------------------
// Simplex cells (sec. 5.1, Tables 11-12: P2 / P3 / P4 triangles with 6 / 12 / 16 integration points
// per cell -- 864/144, 816/68, 384/24).  Reference triangle (0,0), (1,0), (0,1); Lagrange basis of degree k on the
// equispaced lattice (i/k, j/k), i + j <= k, local order j-major: phi = P_i(xi) P_j(eta) P_l(1 - xi - eta), l = k - i - j,
// P_n(t) = prod_{m<n} (k t - m)/(m + 1).  Quadrature: the symmetric rules of degree 4, 6, 8 with exactly those point counts
// (Dunavant 1985), weights normalised to the reference area 1/2.
// ---------------------------------------------------------------------------------------------
void simplex_p(int k, int n, ld t, ld* v, ld* d) {
  ld val = 1, der = 0;
  for (int m = 0; m < n; m++) {
    // product rule, factor (k t - m)/(m + 1)
    der = der * (k * t - m) / (m + 1) + val * k / (ld)(m + 1);
    val = val * (k * t - m) / (m + 1);
  }
  *v = val;
  *d = der;
}

void simplex_rule(int k, std::vector<ld>& xi, std::vector<ld>& eta, std::vector<ld>& w) {
  auto orbit3 = [&](ld a, ld wt) {  // (a, a, 1 - 2a) and permutations
    const ld b = 1 - 2 * a;
    const ld p[3][2] = {{a, a}, {a, b}, {b, a}};
    for (int i = 0; i < 3; i++) {
      xi.push_back(p[i][0]);
      eta.push_back(p[i][1]);
      w.push_back(wt / 2);
    }
  };
  auto orbit6 = [&](ld a, ld b, ld wt) {
    const ld c = 1 - a - b;
    const ld p[6][2] = {{a, b}, {b, a}, {a, c}, {c, a}, {b, c}, {c, b}};
    for (int i = 0; i < 6; i++) {
      xi.push_back(p[i][0]);
      eta.push_back(p[i][1]);
      w.push_back(wt / 2);
    }
  };
  if (k == 2) {  // degree 4, 6 points
    orbit3(0.445948490915965L, 0.223381589678011L);
    orbit3(0.091576213509771L, 0.109951743655322L);
  } else if (k == 3) {  // degree 6, 12 points
    orbit3(0.249286745170910L, 0.116786275726379L);
    orbit3(0.063089014491502L, 0.050844906370207L);
    orbit6(0.053145049844817L, 0.310352451033784L, 0.082851075618374L);
  } else {  // degree 8, 16 points
    xi.push_back(1 / (ld)3);
    eta.push_back(1 / (ld)3);
    w.push_back(0.144315607677787L / 2);
    orbit3(0.459292588292723L, 0.095091634267285L);
    orbit3(0.170569307751760L, 0.103217370534718L);
    orbit3(0.050547228317031L, 0.032458497623198L);
    orbit6(0.008394777409958L, 0.263112829634638L, 0.027230314174435L);
  }
}

// O5  field values at the integration points of one species: f, df/dr, df/dz.
void fields_at_ips(const Problem& pb, const Grid& g, const double* fdof, std::vector<ld>& f,
                   std::vector<ld>& fr, std::vector<ld>& fz) {
  int nip = g.n_ip();
  f.assign(nip, 0);
  fr.assign(nip, 0);
  fz.assign(nip, 0);
  for (size_t e = 0; e < g.cells.size(); e++) {
    std::vector<ld> fe(pb.nb, 0);  // (P_e f)_a
    for (int a = 0; a < pb.nb; a++)
      for (const auto& dw : g.P[e][a]) fe[a] += dw.second * (ld)fdof[dw.first];
    for (int q = 0; q < pb.nq; q++) {
      ld v = 0, vx = 0, ve = 0;
      for (int a = 0; a < pb.nb; a++) {
        v += pb.B[q * pb.nb + a] * fe[a];
        vx += pb.dBxi[q * pb.nb + a] * fe[a];
        ve += pb.dBeta[q * pb.nb + a] * fe[a];
      }
      f[e * pb.nq + q] = v;
      grad_phys(g, (int)e, (int)(e * pb.nq + q), vx, ve, &fr[e * pb.nq + q], &fz[e * pb.nq + q]);
    }
  }
}

// O7  inner integrals and species combination.  Output per species alpha at the IPs of its grid:
//     D_alpha = (Drr, Drz, Dzz), K_alpha = (Kr, Kz).
struct DK {
  std::vector<ld> Drr, Drz, Dzz, Kr, Kz;
};

void inner_integral(const Problem& pb, const double* fentry, std::vector<DK>& dk) {
  const int S = (int)pb.species.size();
  std::vector<std::vector<ld>> f(S), fr(S), fz(S);
  for (int b = 0; b < S; b++)
    fields_at_ips(pb, pb.grids[pb.species[b].grid], fentry + pb.f_off[b], f[b], fr[b], fz[b]);
  dk.assign(S, DK());
  for (int a = 0; a < S; a++) {
    int n = pb.grids[pb.species[a].grid].n_ip();
    dk[a].Drr.assign(n, 0);
    dk[a].Drz.assign(n, 0);
    dk[a].Dzz.assign(n, 0);
    dk[a].Kr.assign(n, 0);
    dk[a].Kz.assign(n, 0);
  }
  for (size_t gi = 0; gi < pb.grids.size(); gi++) {
    const Grid& Gi = pb.grids[gi];
    const int ni = Gi.n_ip();
#pragma omp parallel for schedule(dynamic, 8) num_threads(pb.threads)
    for (int i = 0; i < ni; i++) {
      // G^D_beta(i) (3 numbers) and G^K_beta(i) (2 numbers) for every beta
      std::vector<ld> GD(3 * S, 0), GK(2 * S, 0);
      for (int b = 0; b < S; b++) {
        const Grid& Gj = pb.grids[pb.species[b].grid];
        const int nj = Gj.n_ip();
        for (int j = 0; j < nj; j++) {
          Tensor2V t;
          if (!tensor_closed(Gi.ip_r[i], Gi.ip_z[i], Gj.ip_r[j], Gj.ip_z[j], &t)) continue;
          ld w = Gj.ip_w[j];
          GD[3 * b + 0] += w * f[b][j] * t.UDrr;
          GD[3 * b + 1] += w * f[b][j] * t.UDrz;
          GD[3 * b + 2] += w * f[b][j] * t.UDzz;
          // UK_rz = UD_rz, UK_zz = UD_zz
          GK[2 * b + 0] += w * (t.UKrr * fr[b][j] + t.UDrz * fz[b][j]);
          GK[2 * b + 1] += w * (t.UKzr * fr[b][j] + t.UDzz * fz[b][j]);
        }
      }
      for (int a = 0; a < S; a++) {
        if (pb.species[a].grid != (int)gi) continue;
        ld ma = pb.species[a].mass;  // m0 = 1
        for (int b = 0; b < S; b++) {
          ld mb = pb.species[b].mass;
          ld nuab = pb.nu[a * S + b];
          dk[a].Drr[i] += nuab / (ma * ma) * GD[3 * b + 0];
          dk[a].Drz[i] += nuab / (ma * ma) * GD[3 * b + 1];
          dk[a].Dzz[i] += nuab / (ma * ma) * GD[3 * b + 2];
          dk[a].Kr[i] += nuab / (ma * mb) * GK[2 * b + 0];
          dk[a].Kz[i] += nuab / (ma * mb) * GK[2 * b + 1];
        }
      }
    }
  }
}

int csr_find(const Grid& g, int I, int J) {
  const int* b = g.colidx.data() + g.rowptr[I];
  const int* e = g.colidx.data() + g.rowptr[I + 1];
  const int* p = std::lower_bound(b, e, J);
  if (p == e || *p != J) {
    fprintf(stderr, "oracle: (%d,%d) not in pattern\n", I, J);
    abort();
  }
  return (int)(p - g.colidx.data());
}

// O8 + O9  element matrices A_e[a][c] = sum_q w_q [ (1/dt) phi_a phi_c + grad phi_a . D grad phi_c
//          - (grad phi_a . K) phi_c ]  and assembly A += P_e^T A_e P_e into CSR values.
//          with_operator = false gives the mass matrix alone (inv_dt = 1).
void assemble_species(const Problem& pb, const Grid& g, const DK* dk, ld inv_dt, bool with_operator, double* vals) {
  std::vector<ld> acc(g.colidx.size(), 0);
  const int nb = pb.nb, nq = pb.nq;
  for (size_t e = 0; e < g.cells.size(); e++) {
    std::vector<ld> Ae(nb * nb, 0);
    for (int q = 0; q < nq; q++) {
      int ip = (int)e * nq + q;
      ld w = g.ip_w[ip];
      for (int a = 0; a < nb; a++) {
        ld pa = pb.B[q * nb + a], par, paz;
        grad_phys(g, (int)e, ip, pb.dBxi[q * nb + a], pb.dBeta[q * nb + a], &par, &paz);
        for (int c = 0; c < nb; c++) {
          ld pc = pb.B[q * nb + c], pcr, pcz;
          grad_phys(g, (int)e, ip, pb.dBxi[q * nb + c], pb.dBeta[q * nb + c], &pcr, &pcz);
          ld v = inv_dt * pa * pc;
          if (with_operator) {
            v += par * (dk->Drr[ip] * pcr + dk->Drz[ip] * pcz) + paz * (dk->Drz[ip] * pcr + dk->Dzz[ip] * pcz);
            v -= (par * dk->Kr[ip] + paz * dk->Kz[ip]) * pc;
          }
          Ae[a * nb + c] += w * v;
        }
      }
    }
    for (int a = 0; a < nb; a++)
      for (const auto& ia : g.P[e][a])
        for (int c = 0; c < nb; c++)
          for (const auto& jc : g.P[e][c]) acc[csr_find(g, ia.first, jc.first)] += ia.second * jc.second * Ae[a * nb + c];
  }
  for (size_t n = 0; n < acc.size(); n++) vals[n] = (double)acc[n];
}

// O10  rhs_alpha[a] = sum_e sum_q w_q [ -grad phi_a . D grad f + (grad phi_a . K) f ]   ( = J[f] f )
void apply_species(const Problem& pb, const Grid& g, const DK& dk, const double* fdof, double* rhs) {
  std::vector<ld> f, fr, fz;
  fields_at_ips(pb, g, fdof, f, fr, fz);
  std::vector<ld> acc(g.n_dof, 0);
  const int nb = pb.nb, nq = pb.nq;
  for (size_t e = 0; e < g.cells.size(); e++) {
    for (int a = 0; a < nb; a++) {
      ld s = 0;
      for (int q = 0; q < nq; q++) {
        int ip = (int)e * nq + q;
        ld par, paz;
        grad_phys(g, (int)e, ip, pb.dBxi[q * nb + a], pb.dBeta[q * nb + a], &par, &paz);
        ld flux_r = dk.Drr[ip] * fr[ip] + dk.Drz[ip] * fz[ip] - dk.Kr[ip] * f[ip];
        ld flux_z = dk.Drz[ip] * fr[ip] + dk.Dzz[ip] * fz[ip] - dk.Kz[ip] * f[ip];
        s -= g.ip_w[ip] * (par * flux_r + paz * flux_z);
      }
      for (const auto& ia : g.P[e][a]) acc[ia.first] += ia.second * s;
    }
  }
  for (int i = 0; i < g.n_dof; i++) rhs[i] = (double)acc[i];
}

}  // namespace

// =================================================================================================
// C interface for ctypes (oracle/oracle.py)
// =================================================================================================
extern "C" {

void orc_gauss_legendre(int n, double* x, double* w) {
  std::vector<ld> xl(n), wl(n);
  gauss_legendre(n, xl.data(), wl.data());
  for (int i = 0; i < n; i++) {
    x[i] = (double)xl[i];
    w[i] = (double)wl[i];
  }
}

void orc_lagrange(int k, double xi, double* val, double* der) {
  std::vector<ld> v(k + 1), d(k + 1);
  lagrange_1d(k, xi, v.data(), d.data());
  for (int c = 0; c <= k; c++) {
    val[c] = (double)v[c];
    der[c] = (double)d[c];
  }
}

// out = {K, E, P0, P1, Dc, Q, P2}
void orc_ellip(double m, double mp, double* out) {
  Ellip e = ellip_agm(m, mp);
  out[0] = (double)e.K;
  out[1] = (double)e.E;
  out[2] = (double)e.P0;
  out[3] = (double)e.P1;
  out[4] = (double)e.Dc;
  out[5] = (double)e.Q;
  out[6] = (double)e.P2;
}

// out = {UDrr, UDrz, UDzz, UKrr, UKzr}; returns 1 if the pair is not coincident
int orc_tensor(double r, double z, double rb, double zb, double* out) {
  Tensor2V t;
  bool ok = tensor_closed(r, z, rb, zb, &t);
  out[0] = (double)t.UDrr;
  out[1] = (double)t.UDrz;
  out[2] = (double)t.UDzz;
  out[3] = (double)t.UKrr;
  out[4] = (double)t.UKzr;
  return ok ? 1 : 0;
}

// out = {UDrr, UDrz, UDzz, UKrr, UKrz, UKzr, UKzz, UDzr}
void orc_tensor_quadrature(double r, double z, double rb, double zb, int nphi, double* out) {
  ld o[8];
  tensor_quadrature(r, z, rb, zb, nphi, o);
  for (int k = 0; k < 8; k++) out[k] = (double)o[k];
}

static Problem* new_problem(int degree, int threads) {
  Problem* pb = new Problem();
  pb->k = degree;
  pb->nq1 = degree + 1;
  pb->nb = (degree + 1) * (degree + 1);
  pb->nq = pb->nq1 * pb->nq1;
  pb->threads = threads > 0 ? threads : 1;
  pb->gx.resize(pb->nq1);
  pb->gw.resize(pb->nq1);
  gauss_legendre(pb->nq1, pb->gx.data(), pb->gw.data());
  pb->B.resize(pb->nq * pb->nb);
  pb->dBxi.resize(pb->nq * pb->nb);
  pb->dBeta.resize(pb->nq * pb->nb);
  for (int q2 = 0; q2 < pb->nq1; q2++)
    for (int q1 = 0; q1 < pb->nq1; q1++) {
      std::vector<ld> v1(degree + 1), d1(degree + 1), v2(degree + 1), d2(degree + 1);
      lagrange_1d(degree, pb->gx[q1], v1.data(), d1.data());
      lagrange_1d(degree, pb->gx[q2], v2.data(), d2.data());
      int q = q1 + pb->nq1 * q2;
      for (int a2 = 0; a2 <= degree; a2++)
        for (int a1 = 0; a1 <= degree; a1++) {
          int a = a1 + (degree + 1) * a2;
          pb->B[q * pb->nb + a] = v1[a1] * v2[a2];
          pb->dBxi[q * pb->nb + a] = d1[a1] * v2[a2];
          pb->dBeta[q * pb->nb + a] = v1[a1] * d2[a2];
        }
    }
  return pb;
}

static Problem* new_problem_simplex(int degree, int threads) {
  Problem* pb = new Problem();
  pb->k = degree;
  pb->nq1 = 0;
  pb->simplex = true;
  pb->nb = (degree + 1) * (degree + 2) / 2;
  simplex_rule(degree, pb->sx, pb->se, pb->sw);
  pb->nq = (int)pb->sw.size();
  pb->threads = threads > 0 ? threads : 1;
  pb->B.resize(pb->nq * pb->nb);
  pb->dBxi.resize(pb->nq * pb->nb);
  pb->dBeta.resize(pb->nq * pb->nb);
  for (int q = 0; q < pb->nq; q++) {
    const ld xi = pb->sx[q], eta = pb->se[q], lam = 1 - xi - eta;
    int a = 0;
    for (int j = 0; j <= degree; j++)
      for (int i = 0; i <= degree - j; i++, a++) {
        ld pi, di, pj, dj, pl, dl;
        simplex_p(degree, i, xi, &pi, &di);
        simplex_p(degree, j, eta, &pj, &dj);
        simplex_p(degree, degree - i - j, lam, &pl, &dl);
        pb->B[q * pb->nb + a] = pi * pj * pl;
        pb->dBxi[q * pb->nb + a] = di * pj * pl - pi * pj * dl;
        pb->dBeta[q * pb->nb + a] = pi * dj * pl - pi * pj * dl;
      }
  }
  return pb;
}

static void finish_problem(Problem* pb, const SpeciesDesc* species, int n_species, const double* nu) {
  pb->species.assign(species, species + n_species);
  pb->nu.resize((size_t)n_species * n_species);
  for (int a = 0; a < n_species; a++)
    for (int b = 0; b < n_species; b++)
      pb->nu[a * n_species + b] =
          nu ? (ld)nu[a * n_species + b]
             : (ld)species[a].charge * species[a].charge * (ld)species[b].charge * species[b].charge;  // reading A3
  long long fo = 0, vo = 0;
  for (int a = 0; a < n_species; a++) {
    pb->f_off.push_back(fo);
    pb->v_off.push_back(vo);
    fo += pb->grids[species[a].grid].n_dof;
    vo += (long long)pb->grids[species[a].grid].colidx.size();
  }
  pb->f_stride = fo;
  pb->v_stride = vo;
}

void* orc_create(const GridDesc* grids, int n_grids, const SpeciesDesc* species, int n_species, int degree,
                 const double* nu, int threads) {
  Problem* pb = new_problem(degree, threads);
  pb->grids.resize(n_grids);
  for (int g = 0; g < n_grids; g++) {
    pb->grids[g].desc = grids[g];
    pb->grids[g].k = degree;
    build_mesh(pb->grids[g]);
    build_ips(*pb, pb->grids[g]);
  }
  finish_problem(pb, species, n_species, nu);
  return pb;
}

// Unstructured grids: grid g has n_vertices[g] vertices (vertices[g]: (r, z) pairs) and n_cells[g] cells
// (cells[g]: vertices_per_cell counter-clockwise vertex ids each; 4: quadrilaterals Qk, 3: triangles Pk).  Returns NULL for an
// inverted cell.
void* orc_create_meshes(int n_grids, const int* n_vertices, const double* const* vertices, const int* n_cells,
                        const int* const* cells, int vertices_per_cell, const SpeciesDesc* species, int n_species,
                        int degree, const double* nu, int threads) {
  if ((vertices_per_cell != 3 && vertices_per_cell != 4) || degree < 2 || degree > 4) return nullptr;
  Problem* pb = vertices_per_cell == 3 ? new_problem_simplex(degree, threads) : new_problem(degree, threads);
  pb->grids.resize(n_grids);
  for (int g = 0; g < n_grids; g++) {
    memset(&pb->grids[g].desc, 0, sizeof(GridDesc));
    pb->grids[g].desc.kind = 2;
    pb->grids[g].k = degree;
    if (!build_unstructured(*pb, pb->grids[g], n_vertices[g], vertices[g], n_cells[g], cells[g])) {
      delete pb;
      return nullptr;
    }
  }
  finish_problem(pb, species, n_species, nu);
  return pb;
}

void orc_destroy(void* h) { delete (Problem*)h; }

void orc_sizes(void* h, int* n_dof, int* nnz, int* n_ip, int* n_cells, long long* f_stride, long long* v_stride) {
  Problem* pb = (Problem*)h;
  for (size_t g = 0; g < pb->grids.size(); g++) {
    n_dof[g] = pb->grids[g].n_dof;
    nnz[g] = (int)pb->grids[g].colidx.size();
    n_ip[g] = pb->grids[g].n_ip();
    n_cells[g] = (int)pb->grids[g].cells.size();
  }
  *f_stride = pb->f_stride;
  *v_stride = pb->v_stride;
}

void orc_dof_coords(void* h, int g, double* rz) {
  const Grid& G = ((Problem*)h)->grids[g];
  if (G.unstructured) {
    for (int i = 0; i < G.n_dof; i++) {
      rz[2 * i] = (double)G.node_r[i];
      rz[2 * i + 1] = (double)G.node_z[i];
    }
    return;
  }
  for (int i = 0; i < G.n_dof; i++) {
    rz[2 * i] = (double)(G.dof_ix[i] * G.ur);
    rz[2 * i + 1] = (double)((ld)G.desc.z_min + G.dof_iz[i] * G.uz);
  }
}

void orc_pattern(void* h, int g, int* rowptr, int* colidx) {
  const Grid& G = ((Problem*)h)->grids[g];
  memcpy(rowptr, G.rowptr.data(), sizeof(int) * G.rowptr.size());
  memcpy(colidx, G.colidx.data(), sizeof(int) * G.colidx.size());
}

void orc_ip_table(void* h, int g, double* r, double* z, double* w) {
  const Grid& G = ((Problem*)h)->grids[g];
  for (int i = 0; i < G.n_ip(); i++) {
    r[i] = (double)G.ip_r[i];
    z[i] = (double)G.ip_z[i];
    w[i] = (double)G.ip_w[i];
  }
}

// f, df/dr, df/dz of species s at the IPs of its grid (one batch entry)
void orc_fields(void* h, const double* fentry, int s, double* f, double* fr, double* fz) {
  Problem* pb = (Problem*)h;
  const Grid& G = pb->grids[pb->species[s].grid];
  std::vector<ld> a, b, c;
  fields_at_ips(*pb, G, fentry + pb->f_off[s], a, b, c);
  for (int i = 0; i < G.n_ip(); i++) {
    f[i] = (double)a[i];
    fr[i] = (double)b[i];
    fz[i] = (double)c[i];
  }
}

// D_alpha, K_alpha at the IPs of alpha's grid, concatenated over species: out[alpha] = [n_ip][5]
// (Drr, Drz, Dzz, Kr, Kz), species blocks back to back.
void orc_inner(void* h, const double* fentry, double* out) {
  Problem* pb = (Problem*)h;
  std::vector<DK> dk;
  inner_integral(*pb, fentry, dk);
  size_t o = 0;
  for (size_t a = 0; a < pb->species.size(); a++) {
    int n = pb->grids[pb->species[a].grid].n_ip();
    for (int i = 0; i < n; i++) {
      out[o++] = (double)dk[a].Drr[i];
      out[o++] = (double)dk[a].Drz[i];
      out[o++] = (double)dk[a].Dzz[i];
      out[o++] = (double)dk[a].Kr[i];
      out[o++] = (double)dk[a].Kz[i];
    }
  }
}

// D, K of species `alpha` at arbitrary field points (r,z)[npts] given ANALYTIC source samples at the IPs:
// fsrc[beta] = [n_ip(g(beta))][3] (f, df/dr, df/dz).  Used by pin P5 (Rosenbluth closed forms).
void orc_inner_at_points(void* h, int alpha, const double* const* fsrc, const double* rz, int npts, double* out) {
  Problem* pb = (Problem*)h;
  const int S = (int)pb->species.size();
  ld ma = pb->species[alpha].mass;
  for (int p = 0; p < npts; p++) {
    ld acc[5] = {0, 0, 0, 0, 0};
    for (int b = 0; b < S; b++) {
      const Grid& Gj = pb->grids[pb->species[b].grid];
      ld mb = pb->species[b].mass, nuab = pb->nu[alpha * S + b];
      ld GD[3] = {0, 0, 0}, GK[2] = {0, 0};
      for (int j = 0; j < Gj.n_ip(); j++) {
        Tensor2V t;
        if (!tensor_closed(rz[2 * p], rz[2 * p + 1], Gj.ip_r[j], Gj.ip_z[j], &t)) continue;
        ld w = Gj.ip_w[j], f = fsrc[b][3 * j], fr = fsrc[b][3 * j + 1], fz = fsrc[b][3 * j + 2];
        GD[0] += w * f * t.UDrr;
        GD[1] += w * f * t.UDrz;
        GD[2] += w * f * t.UDzz;
        GK[0] += w * (t.UKrr * fr + t.UDrz * fz);
        GK[1] += w * (t.UKzr * fr + t.UDzz * fz);
      }
      for (int c = 0; c < 3; c++) acc[c] += nuab / (ma * ma) * GD[c];
      for (int c = 0; c < 2; c++) acc[3 + c] += nuab / (ma * mb) * GK[c];
    }
    for (int c = 0; c < 5; c++) out[5 * p + c] = (double)acc[c];
  }
}

// CSR values of M/dt - J for every species of one batch entry: vals[alpha] = [nnz_g(alpha)], back to back.
// dt = +inf gives -J.
void orc_jacobian(void* h, const double* fentry, double dt, double* vals) {
  Problem* pb = (Problem*)h;
  std::vector<DK> dk;
  inner_integral(*pb, fentry, dk);
  ld inv_dt = std::isinf(dt) ? 0 : 1 / (ld)dt;
  for (size_t a = 0; a < pb->species.size(); a++)
    assemble_species(*pb, pb->grids[pb->species[a].grid], &dk[a], inv_dt, true, vals + pb->v_off[a]);
}

// rhs = J[f] f for every species of one batch entry, same layout as f.
void orc_apply(void* h, const double* fentry, double* rhs) {
  Problem* pb = (Problem*)h;
  std::vector<DK> dk;
  inner_integral(*pb, fentry, dk);
  for (size_t a = 0; a < pb->species.size(); a++)
    apply_species(*pb, pb->grids[pb->species[a].grid], dk[a], fentry + pb->f_off[a], rhs + pb->f_off[a]);
}

// CSR values of the mass matrix of grid g.
void orc_mass(void* h, int g, double* vals) {
  Problem* pb = (Problem*)h;
  assemble_species(*pb, pb->grids[g], nullptr, 1, false, vals);
}

// cell rectangles (r0, z0, hr, hz) of grid g, for mesh pins.
void orc_cells(void* h, int g, double* rect) {
  const Grid& G = ((Problem*)h)->grids[g];
  for (size_t e = 0; e < G.cells.size(); e++) {
    ld hr, hz;
    cell_sizes(G, (int)e, &hr, &hz);
    rect[4 * e] = (double)(G.cells[e].ix * G.ur);
    rect[4 * e + 1] = (double)((ld)G.desc.z_min + G.cells[e].iz * G.uz);
    rect[4 * e + 2] = (double)hr;
    rect[4 * e + 3] = (double)hz;
  }
}

}  // extern "C"
