// host_setup.hpp -- host-side set-up of the Landau context (step a0 of DESIGN.md): meshes, dof numbering with
// hanging-node constraints, integration-point tables, CSR pattern and the gather tables the device kernels
// walk.  Runs once in landau_create (the paper also sets grids up on the CPU).
// Independent of oracle/ (no shared code, tables or headers).
#pragma once
#include <string>
#include <vector>

#include "../../include/landau.h"

namespace landau {

// K3 (element matrices + assembly) schedule constants, shared by host set-up and the kernel:
// cells are processed in panels of K3_PC cells (cell order); each element matrix occupies K3_RS doubles of a
// shared-memory ring (a pool of k3_rc matrix positions), entry (a, c) at  k3_entry_offset(a2 n1 + c2, a1 n1 + c1)  (a = a1 + n1 a2, c = c1 + n1 c2).
constexpr int K3_PC = 8;
constexpr int K3_RS = 256;
// offset of entry (n = a2 n1 + c2, m = a1 n1 + c1) inside one element matrix: row n, column m XOR-swizzled by n so that
// the DMMA C-fragment stores of a warp (lanes differ in n / 2 and in m) fall on 32 distinct doubles
#ifdef __CUDACC__
__host__ __device__
#endif
constexpr int k3_entry_offset(int n, int m) { return n * 16 + (m ^ (((n >> 1) & 3) << 2)); }
constexpr int K3_RING_MAX_BYTES = 220 * 1024;
constexpr int K3_NBITS = 17;  // bits of (slot - step base) in a packed single-contribution word

struct HostGrid {
  landau_grid_desc desc;
  int k = 0, nb = 0, nq = 0;
  int n_cells = 0, n_dof = 0, n_ip = 0, nnz = 0;
  // cell rectangles
  std::vector<double> cell_r0, cell_z0, cell_hr, cell_hz;
  // integration points, cell-major (ip = cell*nq + q, q = q1 + (k+1) q2)
  std::vector<double> ip_r, ip_z, ip_w;
  // unstructured meshes only: J^-T at every integration point, [ip][4], (d/dr, d/dz) = gm (d/dxi, d/deta); empty otherwise
  std::vector<double> ip_gm;
  std::vector<double> dof_r, dof_z;
  // element-node -> dof expansion (rows of P_e): entries en_ptr[cell*nb+a] .. en_ptr[cell*nb+a+1]
  std::vector<int> en_ptr, en_dof;
  std::vector<double> en_w;
  // CSR pattern; diag[i] = position of the diagonal entry of row i in colidx / the value array
  std::vector<int> rowptr, colidx, diag;
  // assembly gather: CSR slot n receives sum over entries as_ptr[n]..as_ptr[n+1] of as_w * A_cell[a][c],
  // as_code = cell*nb*nb + a*nb + c
  std::vector<int> as_ptr, as_code;
  std::vector<double> as_w;
  // K3 ring schedule: step s computes cells [s K3_PC, (s+1) K3_PC) into ring positions cell_pos[cell] (< k3_rc; a
  // position is reused once the last slot fed by its matrix has been emitted; halo_begin[s] = first step a CTA that
  // starts emitting at step s must recompute to have every live matrix in its ring) and then
  // emits the CSR slots whose last contributing cell lies in that panel, from three lists (each ascending in n):
  //   em1[em_ptr[s] ..)            one contribution, weight 1:   word = ring offset << K3_NBITS | (n - em_base[s])
  //   em4[em_ptr[S1 + s] ..)       2..4 contributions, all weight 1: {n - base, off0 | off1 << 16, off2 | off3 << 16, 0}
  //                                (unused offsets point at the zero pad behind the ring, offset k3_rc * K3_RS)
  //   emg[em_ptr[2 S1 + s] ..)     anything else (hanging-node weights): n, walks as_ptr / as_roff / as_w
  // with S1 = k3_nsteps + 1.  k3_rc == 0: no ring schedule (ring too large for shared memory or offsets too wide
  // for the packed words), the slot-gather kernel is used for this grid.
  int k3_rc = 0, k3_nsteps = 0;
  std::vector<int> em_ptr, em_base, emg, as_roff, cell_pos, halo_begin;
  std::vector<unsigned> em1, em4;
  // apply gather: dof i receives sum of ap_w * r_cell[a], ap_code = cell*nb + a
  std::vector<int> ap_ptr, ap_code;
  std::vector<double> ap_w;
};

struct HostTables {
  int k = 0, nq1 = 0, nb = 0, nq = 0;
  bool simplex = false;                  // triangles: nb = (k+1)(k+2)/2, reference points (sx, se) and weights sw (sum 1/2)
  std::vector<double> sx, se, sw;
  std::vector<double> gauss_x, gauss_w;  // on [-1,1]
  std::vector<double> B, dBxi, dBeta;    // [q][a]
  std::vector<double> lag_v, lag_d;      // 1-D Lagrange values / derivatives at the Gauss points, [q1][c]
  // constant DMMA A-fragments of K3 (see k3_ring.cuh): [16][32 lanes]; 0..7 = z-direction tables (ztab*2 + mt),
  // 8..15 = r-direction tables ((nt*2 + h)*2 + mt2)
  std::vector<double> k3_frag;
};

// Fills tables for degree k (2 or 3).  Returns false with msg on unsupported degree.
bool build_tables(int k, HostTables* t, std::string* msg);
// Tables of the Pk triangle (k = 2, 3, 4): basis on the equispaced lattice, symmetric rule of degree 2k.
bool build_tables_simplex(int k, HostTables* t, std::string* msg);

// Builds one grid.  status: 0 ok, LANDAU_INVALID_ARG / LANDAU_UNSUPPORTED with msg.
int build_grid(const landau_grid_desc& d, const HostTables& t, HostGrid* g, std::string* msg);
// Builds one unstructured quadrilateral mesh grid (include/landau.h, landau_mesh_desc).
int build_mesh_grid(const landau_mesh_desc& m, const HostTables& t, HostGrid* g, std::string* msg);
// CSR pattern, gather tables and K3 schedule from the element expansions (called by both builders).
int finish_grid(const HostTables& t, HostGrid* g, std::string* msg);

}  // namespace landau
