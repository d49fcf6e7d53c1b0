// host_setup3v.hpp -- host-side set-up of the 3V Landau context (step a0 for the 3V variant): octree
// of Q2 hexahedra on [-half, half]^3 refined about the origin, dof numbering with hanging-face / hanging-edge
// constraints, integration points, CSR pattern and the gather tables the device kernels walk.
// Independent of oracle/ (no shared code, tables or headers): leaves are addressed by (level, i, j, k) in a hash map and the
// leaves whose closure holds a lattice point are found by look-up per level, not by scanning cells.
#pragma once
#include <string>
#include <vector>

#include "../../include/landau3v.h"

namespace landau3v {

constexpr int NB = 27;  // Q2 hexahedron: 3 x 3 x 3 nodes, a = a1 + 3 a2 + 9 a3
constexpr int NQ = 27;  // 3 x 3 x 3 Gauss points, q = q1 + 3 q2 + 9 q3

struct HostGrid3 {
  landau3v_grid_desc desc;
  int n_cells = 0, n_dof = 0, n_ip = 0, nnz = 0;
  std::vector<double> cell_h;            // edge length per cell
  std::vector<double> ip_x, ip_y, ip_z, ip_w;  // cell-major, ip = cell * 27 + q
  std::vector<double> dof_xyz;           // [n_dof][3]
  // element-node -> dof expansion (rows of P_e)
  std::vector<int> en_ptr, en_dof;
  std::vector<double> en_w;
  std::vector<int> rowptr, colidx, diag;
  // assembly gather: CSR slot n = sum over as_ptr[n] .. as_ptr[n+1] of as_w * A_cell[a][c], as_code = (cell * 27 + a) * 27 + c
  std::vector<int> as_ptr, as_code;
  std::vector<double> as_w;
  // apply gather: dof i = sum of ap_w * r_cell[a], ap_code = cell * 27 + a
  std::vector<int> ap_ptr, ap_code;
  std::vector<double> ap_w;
};

struct HostTables3 {
  double gauss_x[3], gauss_w[3];
  std::vector<double> B, dBx, dBy, dBz;  // [q][a], reference derivatives
};

void build_tables3(HostTables3* t);
int build_grid3(const landau3v_grid_desc& d, const HostTables3& t, HostGrid3* g, std::string* msg);

}  // namespace landau3v
