/* landau3v.h -- C ABI of the 3V variant of the batched Landau Jacobian library (same liblandau_b200.so).
 *
 * the hot path of landau.h in full three-dimensional velocity space ("The Landau integral is
 * inherently three dimensional ... Both the 2V and full 3V models are investigated", sec. 2.3; workload of
 * "4 x 4 x 4 initial grid ... 120 (Q2 elements) in 3V ... 1,045 equations with an average of 54.0
 * non-zeros per row"; Tables 6, 14, 16).  For every batch entry and every integration point i of every grid
 *
 *     D_a(i) = sum_b nu_ab (m0/m_a)^2       sum_j w_j f_b(j)            U(v_i, v_j)     (symmetric 3 x 3)
 *     K_a(i) = sum_b nu_ab (m0/m_a)(m0/m_b) sum_j w_j U(v_i, v_j) . grad f_b(j)         (3-vector)
 *     U(v, vb) = (|u|^2 I - u u^T) / |u|^3,  u = v - vb
 *
 * followed by the element matrices of the weak form (eq. 2.4) on Q2 hexahedra and their assembly into the
 * batched CSR of M/dt - J, and the operator application J[f] f.
 *
 * Conventions are those of landau.h (plain C, FP64 / int32, status codes of landau_status, asynchronous on `cuda_stream`,
 * no CPU fallback, contexts not re-entrant).  Discretisation: cubes [-half_width, half_width]^3 of n^3 cells; for
 * l = 1..levels every level-(l-1) cell whose closure contains the origin is split in eight ("one level of AMR refinement
 * about the origin"; n = 4, levels = 1 gives the paper's 120 cells); tri-quadratic Lagrange elements on
 * equispaced nodes, 3 x 3 x 3 Gauss-Legendre points, weights w = gw gw gw h^3 / 8 (Cartesian: no 2 pi, no r); nodes hanging
 * on a coarse face or edge are constrained to that cell's trace; natural boundaries; coincident points
 * (|u|^2 <= 1e-20 (|v|^2 + |vb|^2)) contribute zero.  Dofs are numbered lexicographically by (z, y, x).
 *
 * Layouts: batch_f[b][a][n_dof(g(a))], out_csr_vals[b][a][nnz(g(a))], out_rhs like batch_f (species-major inside an entry,
 * PAPER.md:75); the CSR pattern of a grid is shared by all its species and all entries, columns ascending within a row.
 */
#ifndef LANDAU3V_B200_H
#define LANDAU3V_B200_H

#include "landau.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct landau3v_ctx landau3v_ctx; /* opaque; owns all device tables and scratch */

typedef struct {
  double half_width; /* the grid covers [-half_width, half_width]^3, in units of v0 */
  int n;             /* base cells per direction */
  int levels;        /* refinements of the cells touching the origin */
} landau3v_grid_desc;

/* Build a context (host set-up + one upload).  grids, species (landau_species_desc of landau.h), nu (n_species^2
 * row-major, symmetric; NULL: q_a^2 q_b^2) are host pointers read during the call.  A rank-one nu takes the path that folds
 * all species of a grid into one source field per entry.  cuda_device < 0 builds a host-only context (geometry queries
 * only; compute calls return LANDAU_CUDA_ERROR).  Errors: LANDAU_INVALID_ARG (null / empty / bad extents, species on a
 * missing grid, non-positive mass), LANDAU_UNSUPPORTED (unresolvable constraint chain, more than 16 species),
 * LANDAU_OUT_OF_MEMORY, LANDAU_CUDA_ERROR; message in landau3v_last_error(NULL). */
int landau3v_create(const landau3v_grid_desc* grids, int n_grids, const landau_species_desc* species, int n_species,
                    const double* nu, int cuda_device, landau3v_ctx** out);
void landau3v_destroy(landau3v_ctx* ctx);

/* Sizes per grid (host arrays of n_grids ints, any may be NULL) and strides (doubles per batch entry). */
int landau3v_sizes(const landau3v_ctx* ctx, int* n_dof, int* nnz, int* n_ip, int* n_cells, long long* f_stride,
                   long long* csr_stride);
/* xyz_host: n_dof x 3 doubles. */
int landau3v_dof_coords(const landau3v_ctx* ctx, int grid, double* xyz_host);
/* Integration points of a grid in the library's own order (host arrays of n_ip doubles, any may be NULL). */
int landau3v_ip_table(const landau3v_ctx* ctx, int grid, double* x_host, double* y_host, double* z_host, double* w_host);
/* CSR pattern: device pointers owned by the context (borrowed), or copied into host arrays (n_dof + 1, nnz ints). */
int landau3v_csr_pattern(const landau3v_ctx* ctx, int grid, const int** rowptr_dev, const int** colidx_dev);
int landau3v_csr_pattern_host(const landau3v_ctx* ctx, int grid, int* rowptr_host, int* colidx_host);

/* M/dt - J[f] for `batch` entries (dt > 0; +inf: -J).  batch_f_dev, out_csr_vals_dev: device, caller-owned. */
int landau3v_jacobian(landau3v_ctx* ctx, const double* batch_f_dev, int batch, double dt, double* out_csr_vals_dev,
                      void* cuda_stream);
/* rhs = J[f] f  (M df/dt = rhs). */
int landau3v_apply(landau3v_ctx* ctx, const double* batch_f_dev, int batch, double* out_rhs_dev, void* cuda_stream);
/* Both from ONE evaluation of the inner integral (what a Newton iteration needs). */
int landau3v_jacobian_apply(landau3v_ctx* ctx, const double* batch_f_dev, int batch, double dt, double* out_csr_vals_dev,
                            double* out_rhs_dev, void* cuda_stream);

/* The steps after the path, as for the 2V variant (landau.h: landau_spmv, landau_solve, landau_step; PAPER.md:75-77,
 * 115-117) on the 3V patterns -- same kernels, same argument meaning: y = A x per (entry, species) block; Jacobi-
 * preconditioned TFQMR, one system per CTA and one launch for the batch (x_dev: initial guess on input; iters_dev /
 * relres_dev: [batch][species] or NULL, negative count = tolerance missed); one backward-Euler step
 * (M/dt - J[u]) delta = M (u^k - u)/dt + J[u] u, u <- u + delta by the quasi-Newton iteration, info_host = 4 doubles or
 * NULL (Newton iterations, last largest relative update, most half-steps of any system, unconverged solves);
 * landau3v_step returns LANDAU_NOT_CONVERGED under the conditions landau_step does (u_dev then holds the last iterate). */
int landau3v_spmv(landau3v_ctx* ctx, const double* csr_vals_dev, const double* x_dev, int batch, double* y_dev,
                  void* cuda_stream);
int landau3v_solve(landau3v_ctx* ctx, const double* csr_vals_dev, const double* rhs_dev, int batch, double rtol, int max_it,
                   double* x_dev, int* iters_dev, double* relres_dev, void* cuda_stream);
int landau3v_step(landau3v_ctx* ctx, double* u_dev, int batch, double dt, double newton_rtol, int max_newton,
                  double lin_rtol, int lin_max_it, double* info_host, void* cuda_stream);

/* Same with HOST buffers (copies inside the call, synchronous on return). */
int landau3v_jacobian_host(landau3v_ctx* ctx, const double* batch_f_host, int batch, double dt, double* out_csr_vals_host,
                           void* cuda_stream);

/* Diagnostics (not part of the product path): frozen coefficients of the last pass, [entry][species][9][n_ip] with
 * components Dxx, Dxy, Dxz, Dyy, Dyz, Dzz, Kx, Ky, Kz (n_entries <= entries of the last pass); stage timing
 * (a1 fields, a2 inner integral, a2b combination, a3+a4 assembly or a5 apply) of the last call when enabled; kernels
 * launched so far; inner-integral kernel choice (0 auto, 1 scalar DFMA, 2 DMMA with persistent CTAs sharing the work evenly,
 * 3 DMMA on a grid with the source range cut into planes -- the first version, kept for A/B measurements); assembly choice (0: element matrices on
 * the MMA pipe + gather, 1: the first version, every CSR slot integrating its own entries -- kept for A/B measurements). */
int landau3v_last_coefficients(landau3v_ctx* ctx, double* dk_host, int n_entries);
int landau3v_set_timing(landau3v_ctx* ctx, int enabled);
int landau3v_last_stage_ms(landau3v_ctx* ctx, float* ms4);
long long landau3v_launch_count(const landau3v_ctx* ctx);
int landau3v_set_inner_kernel(landau3v_ctx* ctx, int which);
int landau3v_set_assembly_kernel(landau3v_ctx* ctx, int which);
int landau3v_set_batch_chunk(landau3v_ctx* ctx, int chunk);

const char* landau3v_last_error(const landau3v_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif
