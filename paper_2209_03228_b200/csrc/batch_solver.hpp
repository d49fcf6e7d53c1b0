// batch_solver.hpp -- host side of the batched solve and of the implicit step (k4_solve.cuh), shared by the 2V and the 3V
// contexts.
//
// A BatchSolver is built from the CSR patterns of a context's grids and the block offsets of its species; it owns the
// pattern views the kernels read, the shared-memory plan of k4_tfqmr and the scratch of the step.  The Landau operator
// enters the step only through a callback (A = M/dt - J[u] and J[u] u from one inner integral), so the same Newton loop
// drives either variant.  Every function returns a landau_status code and leaves a message in `err`.
#pragma once
#include <cuda_runtime.h>

#include <functional>
#include <string>
#include <vector>

namespace landau {

struct SolverGridView {
  int n, nnz;
  const int *d_rowptr, *d_colidx;  // device, owned by the context
  const int* h_diag;               // host: position of a_ii in the value array, n entries
};
struct SolverSpeciesView {
  int grid;
  long long f_off, v_off;
};

struct BatchSolver {
  int device = -1, S = 0, max_n = 0, smem_n = 0, mat_nnz = 0;
  size_t smem = 0;
  int warp_wpc = 0, warp_n = 0, warp_nnz = 0;  // warp-per-system mode of small systems: warps per CTA, padded sizes
  size_t warp_smem = 0;
  bool use_warp = false;  // opt-in (A/B): one warp per system where it applies; measured slower than one CTA per system
  long long f_stride = 0, v_stride = 0;
  void *d_grid = nullptr, *d_spec = nullptr;  // K4Grid[G], K4Species[S]
  std::vector<void*> allocs;
  double *ws = nullptr, *A = nullptr, *vec = nullptr, *misc = nullptr;  // TFQMR workspace; scratch of the step
  size_t ws_cap = 0, A_cap = 0, vec_cap = 0, misc_cap = 0;
  long long launches = 0;
  std::string err;
};

int solver_create(BatchSolver& s, int device, const std::vector<SolverGridView>& grids,
                  const std::vector<SolverSpeciesView>& species, long long f_stride, long long v_stride);
void solver_destroy(BatchSolver& s);

// y = A x for every (entry, species) block; vals_stride = 0 applies ONE set of values (e.g. the mass matrix) to all entries
int solver_spmv(BatchSolver& s, const double* vals, long long vals_stride, const double* x, int batch, double* y,
                cudaStream_t st);
// Jacobi-preconditioned TFQMR, one system per CTA, one launch; iters[b * S + a] < 0: not converged (-(half-steps) - 1)
int solver_tfqmr(BatchSolver& s, const double* vals, const double* rhs, int batch, double rtol, int max_it, double* x,
                 int* iters, double* relres, cudaStream_t st);

// The same solve for callers that may not allocate (landau.h: landau_solve_noalloc): the global Krylov workspace of systems
// too large for shared memory is a fixed static __device__ array of batch_solver.cu instead of s.ws, so no cudaMalloc is
// ever issued; LANDAU_INVALID_ARG when batch * S systems of 7 max_n doubles exceed it.  One array per device, shared by
// every caller: overlapping calls race.  The first call on a device looks up the array's address (before any capture).
int solver_tfqmr_noalloc(BatchSolver& s, const double* vals, const double* rhs, int batch, double rtol, int max_it, double* x,
                         int* iters, double* relres, cudaStream_t st);

// A = M/dt - J[u] (CSR values) and ju = J[u] u for `batch` entries, both from one inner integral, on the step's stream
using JacobianApplyFn = std::function<int(const double* u, int batch, double dt, double* A, double* ju)>;

// One backward-Euler step  M (u1 - u0)/dt = J[u1] u1  by the quasi-Newton iteration on the sparse Jacobian:
// per iteration one Jacobian + operator application, the mass product, one batched TFQMR solve and the update with its norm;
// one stream synchronisation per iteration.  info_host (4 doubles, may be NULL): Newton iterations, last max relative
// update, worst TFQMR half-step count, number of unconverged linear solves.
int solver_step(BatchSolver& s, const JacobianApplyFn& jacobian_apply, const double* mass_vals, double* u, int batch, double dt,
                double newton_rtol, int max_newton, double lin_rtol, int lin_max_it, double* info_host, cudaStream_t st);

}  // namespace landau
