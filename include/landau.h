/* landau.h -- C ABI of the B200-native batched Landau Jacobian library (liblandau_b200.so).
 *
 * One thing is built here: the data-parallel hot path of the fully implicit Landau collision advance of
 * arxiv 2209.03228 -- for every batch entry (an independent axisymmetric (r,z) velocity-space
 * problem, sec. 3.1) the O(N^2) inner integral of the Landau tensor (eq. 2.1/2.3),
 * the per-element finite-element matrices of the weak form (eq. 2.4) and the assembly of the
 * shifted matrix M/dt - J into one batched CSR per species.
 *
 * Conventions common to every entry point
 *   - plain C: pointers + sizes, no C++/torch types.  "host" / "dev" in a parameter comment says where the
 *     memory lives.  Device pointers must belong to the CUDA device the context was created on.
 *   - all floating point is IEEE FP64, all indices int32 (offsets into batched arrays: long long).
 *   - return value: 0 (LANDAU_OK) or a negative landau_status; nothing throws, nothing aborts.  A message for
 *     the last failure of a context is kept in landau_last_error(ctx) (ctx == NULL: last create failure).
 *   - a context is owned by the caller (landau_destroy), is bound to one device, and is not re-entrant:
 *     calls on one context must be serialised by the caller.  Different contexts are independent.
 *   - landau_jacobian / landau_apply are asynchronous on `cuda_stream` (a cudaStream_t passed as void*; NULL =
 *     legacy default stream) and perform no hidden device synchronisation unless their scratch must grow
 *     (first call with a larger batch: one cudaMalloc; landau_reserve pre-sizes it).  Stages are bracketed by NVTX
 *     ranges ("landau K1 ..", "landau K2 ..", ...).
 *   - diagnostics, probes and tuning knobs (not part of the product ABI) are declared in landau_debug.h.
 *   - there is no CPU fallback: without a CUDA device landau_create fails with LANDAU_CUDA_ERROR.
 *
 * Units and discretisation (readings A3-A17): velocity coordinates of every grid are in the common
 * unit v0 (electron thermal speed), m0 = electron mass = 1, f in units n0/v0^3; tensor-product Lagrange Qk
 * elements on k+1 equispaced nodes, (k+1)^2 Gauss-Legendre points per cell, axis-aligned rectangular cells,
 * hanging nodes of quadtree grids constrained to the coarse edge, natural (zero-flux) boundaries, no
 * essential boundary conditions; coincident integration points contribute zero to the inner integral.
 */
#ifndef LANDAU_B200_H
#define LANDAU_B200_H

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  LANDAU_OK = 0,
  LANDAU_INVALID_ARG = -1,   /* NULL pointer, non-positive size, dt <= 0, species on a missing grid, ...   */
  LANDAU_UNSUPPORTED = -2,   /* degree not in {2,3,4}, n_gauss_1d != degree+1, grid kind unknown, chain of
                                hanging-node constraints (mesh not 2:1 balanced)                           */
  LANDAU_OUT_OF_MEMORY = -3, /* host or device allocation failed                                           */
  LANDAU_CUDA_ERROR = -4,    /* any other CUDA runtime failure (no device, launch failure, ...)            */
  LANDAU_NOT_CONVERGED = -5  /* landau_step / landau3v_step only: the state was advanced to the last Newton
                                iterate, which is not the step's solution (see landau_step)                */
} landau_status;

typedef struct landau_ctx landau_ctx; /* opaque; owns all device tables and scratch */

/* One velocity-space grid: the half plane r in [0,r_max], z in [z_min,z_max] (sec. 2.3).
 * kind 0: uniform nr x nz cells.  kind 1: quadtree: base nr x nz cells; for l = 1..levels every
 * level-(l-1) cell inside the box [0, r_max/2^l] x [zc - zh/2^l, zc + zh/2^l] (zc, zh = centre and half extent
 * of the z range) is split in four (reading A12). */
typedef struct {
  int kind;
  double r_max, z_min, z_max;
  int nr, nz;
  int levels; /* ignored for kind 0 */
} landau_grid_desc;

/* One species: mass in units of m0 (electron mass), charge in units of e, index of the grid it lives on.
 * Several species may share a grid (sec. 3). */
typedef struct {
  double mass, charge;
  int grid;
} landau_species_desc;

/* Element degree k (Qk, k = 2, 3, 4 -- the degrees of PAPER.md:309-313 Table 13) and Gauss points per direction (must be
 * k+1).  Q4 cells (25 basis functions) take the general element-matrix + gather assembly, Q2 / Q3 the ring kernel. */
typedef struct {
  int degree;
  int n_gauss_1d;
} landau_quadrature_desc;

/* Build a context: meshes, dof numbering (lexicographic by (z,r)), hanging-node constraints, integration
 * point tables, CSR patterns and gather tables, uploaded once to `cuda_device`.
 *   grids[n_grids], species[n_species], quadrature : host, read only during the call.
 *   nu : host, n_species x n_species row-major symmetric collision-frequency matrix nu~_ab of eq. (2.2)
 *        (PAPER.md:52-57), or NULL for nu_ab = q_a^2 q_b^2 (equal Coulomb logarithms, reading A3).
 *        A matrix of the form a_a * b_b is detected and takes the fast path that sums the species of all
 *        grids into one source field per batch entry before the inner integral.
 *   cuda_device : CUDA device ordinal.  A NEGATIVE value builds a host-only context: the geometry queries
 *        (landau_sizes, landau_dof_coords, landau_ip_table, landau_csr_pattern_host) work without a GPU, every
 *        compute entry point returns LANDAU_CUDA_ERROR -- used by the CPU-only test-suite for the host logic.
 *   out : receives the context; untouched on failure. */
int landau_create(const landau_grid_desc* grids, int n_grids, const landau_species_desc* species, int n_species,
                  const landau_quadrature_desc* quadrature, const double* nu, int cuda_device, landau_ctx** out);

/* One unstructured velocity-space grid of straight-sided quadrilaterals on the (r, z) half plane (PAPER.md:225-229
 * sec. 5.2, "unstructured grids with ... tensor elements").  The mesh must be conforming (no hanging
 * nodes); every cell lists its four vertices counter-clockwise (positive Jacobian).  The cell geometry is the bilinear
 * map of the reference square, so the gradient transformation J^-T and det J differ from point to point; Qk nodes are
 * the images of the equispaced reference nodes. */
typedef struct {
  int n_vertices;
  const double* vertices_rz; /* host, n_vertices x 2: (r, z) in units of v0 */
  int n_cells;
  const int* cells;          /* host, n_cells x vertices_per_cell vertex indices, counter-clockwise */
  int vertices_per_cell;     /* 4: quadrilaterals (Qk, k = 2, 3, 4); 3: triangles (Pk, k = 2, 3, 4; sec. 5.1) */
} landau_mesh_desc;

/* landau_create for unstructured quadrilateral grids: meshes[n_grids] (host, read during the call) take the place of the
 * grid descriptors, everything else as above.  Dofs are ordered by (z, r) of their coordinates (on a grid of 2^-30 of the
 * mesh extent), exposed through landau_dof_coords; all other entry points work unchanged on such a context.
 * landau_last_coefficients (landau_debug.h) returns the coefficients pulled back to the reference cell on these grids.
 * Triangles: Lagrange Pk on the equispaced lattice of the cell, the symmetric quadrature rule of degree 2k with 6 / 12 / 16
 * points (the point counts of the paper's Tables 11-12), affine geometry; `quadrature->n_gauss_1d` must still be degree + 1
 * and is otherwise ignored; all meshes of a context must have the same cell type.
 * Extra errors: LANDAU_INVALID_ARG for a cell with a missing vertex or a non-positive Jacobian, LANDAU_UNSUPPORTED for
 * mixed cell types or a degree the cell type does not have. */
int landau_create_meshes(const landau_mesh_desc* meshes, int n_grids, const landau_species_desc* species, int n_species,
                         const landau_quadrature_desc* quadrature, const double* nu, int cuda_device, landau_ctx** out);

/* Frees every host and device resource of the context (synchronises the device first).  NULL is a no-op. */
void landau_destroy(landau_ctx* ctx);

/* Sizes.  Arrays have one entry per grid (host, may be NULL to skip):
 *   n_dof[g]  unknowns (equations) of one species on grid g,
 *   nnz[g]    structural nonzeros of grid g's CSR pattern,
 *   n_ip[g]   integration points of grid g,
 *   n_cells[g] cells of grid g.
 *   f_stride   doubles per batch entry of batch_f / out_rhs  = sum over species a of n_dof[grid(a)],
 *   csr_stride doubles per batch entry of out_csr_vals       = sum over species a of nnz[grid(a)]. */
int landau_sizes(const landau_ctx* ctx, int* n_dof, int* nnz, int* n_ip, int* n_cells, long long* f_stride,
                 long long* csr_stride);

/* (r,z) of every dof of grid g, in dof order: rz_host[2*i] = r, rz_host[2*i+1] = z   (host, n_dof[g] x 2). */
int landau_dof_coords(const landau_ctx* ctx, int grid, double* rz_host);

/* (r, z, w) of the integration points of grid g (host arrays of n_ip[g]; any may be NULL).
 * w = Gauss weight x cell Jacobian x r (cylindrical measure, the common 2 pi dropped; reading A6). */
int landau_ip_table(const landau_ctx* ctx, int grid, double* r_host, double* z_host, double* w_host);

/* CSR pattern of grid g, shared by every species on the grid and every batch entry.  The pointers are DEVICE
 * pointers owned by the context (valid until landau_destroy): rowptr[n_dof+1], colidx[nnz], columns ascending
 * in each row, structural (every pair of dofs coupled by a cell, including parent-edge couplings of hanging
 * nodes).  landau_csr_pattern_host copies the same arrays into caller-owned host memory. */
int landau_csr_pattern(const landau_ctx* ctx, int grid, const int** rowptr_dev, const int** colidx_dev);
int landau_csr_pattern_host(const landau_ctx* ctx, int grid, int* rowptr_host, int* colidx_host);

/* The batched shifted Jacobian  M/dt - J[f]  (sparse, inner integrals frozen: PAPER.md:73).
 *   batch_f_dev      : dev, [batch][species a][n_dof[grid(a)]]   nodal values (the paper's u = [f_1..f_S])
 *   dt               : > 0; +infinity gives the unshifted -J
 *   out_csr_vals_dev : dev, [batch][species a][nnz[grid(a)]]     every entry written exactly once
 * J_ac = sum_q w_q [ -grad phi_a . D_a grad phi_c + (grad phi_a . K_a) phi_c ],  M_ac = sum_q w_q phi_a phi_c,
 * D_a = sum_b nu_ab (m0/m_a)^2 INT U fb,  K_a = sum_b nu_ab (m0/m_a)(m0/m_b) INT U . grad fb   (eq. 2.1, 2.3).
 * batch == 0 is a successful no-op. */
int landau_jacobian(landau_ctx* ctx, const double* batch_f_dev, int batch, double dt, double* out_csr_vals_dev,
                    void* cuda_stream);

/* Operator application  rhs = J[f] f  (so that M df/dt = rhs; residual of the Newton iteration).
 *   out_rhs_dev : dev, same layout as batch_f_dev. */
int landau_apply(landau_ctx* ctx, const double* batch_f_dev, int batch, double* out_rhs_dev, void* cuda_stream);

/* Batched CSR product  y = A x  for every (entry, species) block of a value array in the layout of out_csr_vals_dev
 * (pattern of the block's grid); x_dev, y_dev in the layout of batch_f_dev.  With the values of M/dt - J and of -J
 * (dt = +inf) it gives the right-hand side (M/dt) f of the implicit step. */
int landau_spmv(landau_ctx* ctx, const double* csr_vals_dev, const double* x_dev, int batch, double* y_dev,
                void* cuda_stream);

/* Batched linear solve  A x = b  of every (entry, species) block, the step that follows the Jacobian construction in
 * the implicit advance (sec. 3.2, 127): TFQMR with Jacobi preconditioning, one system per thread
 * block, the whole batch in one launch (reading A18 for the iteration the paper only cites).
 *   csr_vals_dev : dev, [batch][species a][nnz[grid(a)]]      e.g. the output of landau_jacobian
 *   rhs_dev      : dev, [batch][species a][n_dof[grid(a)]]
 *   x_dev        : dev, same layout; ON INPUT the initial guess (zeros are fine), on output the solution
 *   rtol         : a run stops when the TFQMR residual bound  tau sqrt(m)  <=  rtol * || D^-1 (b - A x0) ||; the true
 *                  Jacobi-scaled residual is then computed and, if it misses the tolerance (the recursive bound drifts
 *                  on ill-conditioned blocks), the iteration restarts from the current x (a run is also restarted after 600 half-steps, which ends stagnation)
 *   max_it       : at most 2 max_it half-steps (max_it products with A beyond the first)
 *   iters_dev    : dev, [batch][species] or NULL: half-steps taken; negative (-m-1) when the tolerance was not reached
 *                  in 2 max_it half-steps or the iteration broke down (x then holds the last iterate)
 *   relres_dev   : dev, [batch][species] or NULL: last residual norm (true if converged, else the bound) relative to
 *                  the initial Jacobi-scaled residual
 * Asynchronous on cuda_stream.  Zero diagonal entries are not supported (Jacobi). */
int landau_solve(landau_ctx* ctx, const double* csr_vals_dev, const double* rhs_dev, int batch, double rtol, int max_it,
                 double* x_dev, int* iters_dev, double* relres_dev, void* cuda_stream);

/* landau_solve for callers that must not allocate device memory.
 *
 * Who that is: a host application that has already handed the GPU's memory to its own pool -- a particle code that sizes
 * its arrays to fill the card, a framework whose caching allocator sits at its limit -- so that a cudaMalloc from inside
 * this library fails or eats the headroom the application counted on; and a time-step loop that cannot afford the
 * device-wide synchronisation a cudaMalloc / cudaFree brings with it.  landau_solve is not safe for them: when a grid has
 * more unknowns than fit in one SM's shared memory (beyond about 4,100; PAPER.md:117 discusses that case) its kernel keeps
 * the seven Krylov vectors of every system in a global-memory workspace, which landau_solve grows with cudaMalloc.
 *
 * This entry point runs the same kernel with that workspace in a fixed array that is part of the library image
 * (LANDAU_SOLVE_NOALLOC_WS_BYTES, a `static __device__` array: every GPU on which the library is used holds it from load
 * to process exit, whether or not this function is ever called).  It calls no cudaMalloc, cudaFree or other allocating
 * routine.  Arguments, layouts, stopping rule and results are those of landau_solve -- bit for bit, the arithmetic is
 * the same; one system per thread block (the landau_set_solve_kernel knob of landau_debug.h is not consulted).
 *
 * Limit: only contexts with such a large grid use the array, 7 * (largest n_dof of the context) doubles per
 * (entry, species) system.  A call with  7 * max n_dof * batch * n_species * 8  >  LANDAU_SOLVE_NOALLOC_WS_BYTES  is refused
 * with LANDAU_INVALID_ARG before anything is launched (landau_last_error names the largest batch that fits): split the
 * batch.  Contexts whose systems all fit in shared memory need no workspace and have no limit.
 *
 * First call on a device: the function asks the runtime once per device for the array's device address (the context's
 * device is made current first).  Make that first call before starting any stream capture.
 * Sharing: there is ONE array per device and process; every call on that device uses it and leaves its vectors behind.
 * Nothing in it has to be zero on entry (the kernel writes each vector before it reads it), so calls in a row need no
 * clearing; but two calls that can run on the GPU at the same time -- different streams, different contexts, different
 * host threads -- overwrite each other's vectors and both results are garbage.  Order them on one stream or with events. */
#define LANDAU_SOLVE_NOALLOC_WS_BYTES (32u << 20) /* 32 MiB = 4,194,304 doubles: 126 systems of 4,753 unknowns */
int landau_solve_noalloc(landau_ctx* ctx, const double* csr_vals_dev, const double* rhs_dev, int batch, double rtol,
                         int max_it, double* x_dev, int* iters_dev, double* relres_dev, void* cuda_stream);

/* Jacobian and operator application from ONE evaluation of the inner integral (what a Newton iteration needs):
 * out_csr_vals_dev as landau_jacobian, out_rhs_dev as landau_apply. */
int landau_jacobian_apply(landau_ctx* ctx, const double* batch_f_dev, int batch, double dt, double* out_csr_vals_dev,
                          double* out_rhs_dev, void* cuda_stream);

/* One backward-Euler step of the implicit collision advance for every batch entry (sec. 2.2), by the
 * quasi-Newton iteration on the sparse frozen-coefficient Jacobian:
 *     (M/dt - J[u]) delta = M (u^k - u)/dt + J[u] u,    u <- u + delta,    starting from u = u^k,
 * until the largest relative update  max over (entry, species) of ||delta|| / ||u||  is <= newton_rtol, at most
 * max_newton iterations; every linear system is solved by landau_solve(lin_rtol, lin_max_it) from a zero guess.
 *   u_dev     : dev, layout of batch_f_dev; ON INPUT u^k, on output u^{k+1}
 *   info_host : host, 4 doubles or NULL: Newton iterations done, last largest relative update, most linear half-steps
 *               any system took, number of linear solves that missed lin_rtol
 * Returns LANDAU_NOT_CONVERGED (with info_host filled and u_dev holding the last iterate) when the update is still above
 * newton_rtol after max_newton iterations, or when a linear solve of the last iteration missed lin_rtol or broke down;
 * linear solves that failed in earlier iterations only cost Newton iterations and are just counted in info_host[3].
 * Every operator application runs in the kernels of this library; the call synchronises cuda_stream once per Newton
 * iteration (to read the update norm).  Scratch (the batch's CSR values and four vectors) is grown on demand. */
int landau_step(landau_ctx* ctx, double* u_dev, int batch, double dt, double newton_rtol, int max_newton, double lin_rtol,
                int lin_max_it, double* info_host, void* cuda_stream);

/* Host-buffer convenience: same as landau_jacobian / landau_apply with HOST pointers (pageable or pinned); the
 * library stages the copies in internal device buffers and synchronises before returning.  landau_jacobian_host
 * cuts the batch into pieces and copies the CSR values of a finished piece to the host on a second (internal)
 * stream while the kernels of the next piece run on `cuda_stream`; results equal the one-piece path up to the
 * summation order of the inner integral (<= 1e-14 relative; bit-identical when the many-column stream mode is off). */
int landau_jacobian_host(landau_ctx* ctx, const double* batch_f_host, int batch, double dt, double* out_csr_vals_host,
                         void* cuda_stream);
int landau_apply_host(landau_ctx* ctx, const double* batch_f_host, int batch, double* out_rhs_host, void* cuda_stream);

/* Pre-size every scratch buffer of landau_jacobian / landau_apply / landau_jacobian_apply for calls with
 * batch <= max_batch (at the current batch chunk), so that those calls neither allocate nor synchronise from the first
 * one on.  Optional: without it the scratch grows on demand (one cudaMalloc + device synchronisation per growth).
 * Covers the element-matrix scratch of species that are not assembled by the ring kernel (under the assembly mode set at
 * the time of the call).  Not covered: the scratch of landau_solve (large systems only; see landau_solve_noalloc), of
 * landau_step and of the *_host variants, which still grow on first use.
 * Synchronises the device.  LANDAU_OUT_OF_MEMORY leaves the context usable. */
int landau_reserve(landau_ctx* ctx, int max_batch);

/* Message of the last failure of `ctx` (ctx == NULL: of the last failed landau_create); owned by the library. */
const char* landau_last_error(const landau_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* LANDAU_B200_H */
