// host_setup.hpp -- host-side set-up of the Landau context (step a0 of DESIGN.md): meshes, dof numbering with
// hanging-node constraints, integration-point tables, CSR pattern and the gather tables the device kernels
// walk.  Runs once in landau_create (the paper also sets grids up on the CPU).
// Independent of oracle/ (no shared code, tables or headers).
#pragma once
#include <string>
#include <vector>

#include "../../include/landau.h"

namespace landau {

struct HostGrid {
  landau_grid_desc desc;
  int k = 0, nb = 0, nq = 0;
  int n_cells = 0, n_dof = 0, n_ip = 0, nnz = 0;
  // cell rectangles
  std::vector<double> cell_r0, cell_z0, cell_hr, cell_hz;
  // integration points, cell-major (ip = cell*nq + q, q = q1 + (k+1) q2)
  std::vector<double> ip_r, ip_z, ip_w;
  std::vector<double> dof_r, dof_z;
  // element-node -> dof expansion (rows of P_e): entries en_ptr[cell*nb+a] .. en_ptr[cell*nb+a+1]
  std::vector<int> en_ptr, en_dof;
  std::vector<double> en_w;
  // CSR pattern
  std::vector<int> rowptr, colidx;
  // assembly gather: CSR slot n receives sum over entries as_ptr[n]..as_ptr[n+1] of as_w * A_cell[a][c],
  // as_code = cell*nb*nb + a*nb + c
  std::vector<int> as_ptr, as_code;
  std::vector<double> as_w;
  // apply gather: dof i receives sum of ap_w * r_cell[a], ap_code = cell*nb + a
  std::vector<int> ap_ptr, ap_code;
  std::vector<double> ap_w;
};

struct HostTables {
  int k = 0, nq1 = 0, nb = 0, nq = 0;
  std::vector<double> gauss_x, gauss_w;  // on [-1,1]
  std::vector<double> B, dBxi, dBeta;    // [q][a]
};

// Fills tables for degree k (2 or 3).  Returns false with msg on unsupported degree.
bool build_tables(int k, HostTables* t, std::string* msg);

// Builds one grid.  status: 0 ok, LANDAU_INVALID_ARG / LANDAU_UNSUPPORTED with msg.
int build_grid(const landau_grid_desc& d, const HostTables& t, HostGrid* g, std::string* msg);

}  // namespace landau
