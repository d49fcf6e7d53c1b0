// batch_solver.cu -- host side of the batched TFQMR solve and of the backward-Euler quasi-Newton step (batch_solver.hpp);
// the kernels are those of k4_solve.cuh, compiled in this translation unit only.
#include "batch_solver.hpp"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <mutex>

#include "../../include/landau.h"
#include "k4_solve.cuh"

namespace landau {
namespace {

int cuda_fail(BatchSolver& s, cudaError_t e, const char* what) {
  s.err = std::string(what) + ": " + cudaGetErrorString(e);
  return e == cudaErrorMemoryAllocation ? LANDAU_OUT_OF_MEMORY : LANDAU_CUDA_ERROR;
}
#define SOLVER_TRY(s, expr)                                   \
  do {                                                        \
    cudaError_t e_ = (expr);                                  \
    if (e_ != cudaSuccess) return cuda_fail(s, e_, #expr);    \
  } while (0)

template <class T>
int upload(BatchSolver& s, const T* h, size_t n, void** out) {
  void* d = nullptr;
  SOLVER_TRY(s, cudaMalloc(&d, sizeof(T) * std::max<size_t>(n, 1)));
  s.allocs.push_back(d);
  if (n) SOLVER_TRY(s, cudaMemcpy(d, h, sizeof(T) * n, cudaMemcpyHostToDevice));
  *out = d;
  return LANDAU_OK;
}

int grow(BatchSolver& s, double** p, size_t* cap, size_t need) {
  if (need <= *cap) return LANDAU_OK;
  if (*p) {
    SOLVER_TRY(s, cudaDeviceSynchronize());
    SOLVER_TRY(s, cudaFree(*p));
    *p = nullptr;
    *cap = 0;
  }
  SOLVER_TRY(s, cudaMalloc(p, need * sizeof(double)));
  *cap = need;
  return LANDAU_OK;
}

// The dynamic shared-memory limit belongs to the device's copy of k4_tfqmr, not to a context: keep a per-device
// high-water mark and only ever raise it, so that live contexts of different sizes can be used alternately.
size_t g_smem_set[64] = {0}, g_smem_set_warp[64] = {0};

}  // namespace

int solver_create(BatchSolver& s, int device, const std::vector<SolverGridView>& grids,
                  const std::vector<SolverSpeciesView>& species, long long f_stride, long long v_stride) {
  s.device = device;
  s.S = (int)species.size();
  s.f_stride = f_stride;
  s.v_stride = v_stride;
  std::vector<K4Grid> kg(grids.size());
  int max_nnz = 0;
  for (size_t g = 0; g < grids.size(); ++g) {
    void* d_diag = nullptr;
    if (int rc = upload(s, grids[g].h_diag, (size_t)grids[g].n, &d_diag)) return rc;
    kg[g] = K4Grid{grids[g].n, grids[g].nnz, grids[g].d_rowptr, grids[g].d_colidx, static_cast<const int*>(d_diag)};
    s.max_n = std::max(s.max_n, grids[g].n);
    max_nnz = std::max(max_nnz, grids[g].nnz);
  }
  std::vector<K4Species> ks(species.size());
  for (size_t a = 0; a < species.size(); ++a) ks[a] = K4Species{species[a].grid, species[a].f_off, species[a].v_off};
  if (int rc = upload(s, kg.data(), kg.size(), &s.d_grid)) return rc;
  if (int rc = upload(s, ks.data(), ks.size(), &s.d_spec)) return rc;
  // Krylov vectors in shared memory when 7 n doubles fit beside the reduction scratch (227 KB per CTA on sm_100)
  const size_t limit = 227 * 1024, fixed = 2 * (K4_THREADS / 32) * sizeof(double);
  s.smem_n = (int)((limit - fixed) / (K4_NVEC * sizeof(double)));
  const int n_in_smem = std::min(s.max_n, s.smem_n);
  s.smem = fixed + (size_t)K4_NVEC * n_in_smem * sizeof(double);
  // small systems: the pattern and one value block also go to shared memory when everything stays below 56 KB
  // (four systems per SM)
  const size_t mat = (size_t)max_nnz * 12 + (size_t)(s.max_n + 2) * 4;
  s.mat_nnz = (s.max_n <= s.smem_n && s.smem + mat <= 56 * 1024) ? max_nnz : 0;
  if (s.mat_nnz) s.smem += mat + K4_NVEC * sizeof(double);  // vectors padded to an even length
  // smaller still: one WARP per system (no block-wide barrier in the iteration), the warps of a CTA on entries of one
  // species sharing its pattern; taken when at least four systems fit in the shared memory of an SM
  {
    const size_t n_even = (size_t)(s.max_n + 1) & ~(size_t)1, nnz_even = (size_t)(max_nnz + 1) & ~(size_t)1;
    const size_t pattern = ((nnz_even + n_even + 2 + 1) / 2) * sizeof(double);
    const size_t per_warp = (K4_NVEC * n_even + nnz_even) * sizeof(double);
    const size_t room = limit > pattern ? limit - pattern : 0;
    const int wpc = (int)std::min<size_t>(room / per_warp, 8);
    if (wpc >= 4) {
      s.warp_wpc = wpc;
      s.warp_n = (int)n_even;
      s.warp_nnz = (int)nnz_even;
      s.warp_smem = pattern + wpc * per_warp;
    }
  }
  size_t* cur = device >= 0 && device < 64 ? &g_smem_set[device] : nullptr;
  if (!cur || s.smem > *cur) {
    SOLVER_TRY(s, cudaFuncSetAttribute(k4_tfqmr_t<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)s.smem));
    if (cur) *cur = s.smem;
  }
  size_t* curw = device >= 0 && device < 64 ? &g_smem_set_warp[device] : nullptr;
  if (s.warp_wpc && (!curw || s.warp_smem > *curw)) {
    SOLVER_TRY(s, cudaFuncSetAttribute(k4_tfqmr_t<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)s.warp_smem));
    if (curw) *curw = s.warp_smem;
  }
  return LANDAU_OK;
}

void solver_destroy(BatchSolver& s) {
  for (void* p : s.allocs) cudaFree(p);
  s.allocs.clear();
  for (double* p : {s.ws, s.A, s.vec, s.misc})
    if (p) cudaFree(p);
  s.ws = s.A = s.vec = s.misc = nullptr;
  s.ws_cap = s.A_cap = s.vec_cap = s.misc_cap = 0;
}

int solver_spmv(BatchSolver& s, const double* vals, long long vals_stride, const double* x, int batch, double* y,
                cudaStream_t st) {
  k4_spmv_batch<<<batch * s.S, K4_THREADS, 0, st>>>(static_cast<const K4Grid*>(s.d_grid), static_cast<const K4Species*>(s.d_spec),
                                                   s.S, vals, vals_stride, x, s.f_stride, y);
  ++s.launches;
  SOLVER_TRY(s, cudaGetLastError());
  return LANDAU_OK;
}

int solver_tfqmr(BatchSolver& s, const double* vals, const double* rhs, int batch, double rtol, int max_it, double* x,
                 int* iters, double* relres, cudaStream_t st) {
  long long ws_stride = 0;
  if (s.max_n > s.smem_n) {  // some grid's vectors do not fit in shared memory: global workspace
    ws_stride = (long long)K4_NVEC * s.max_n;
    if (int rc = grow(s, &s.ws, &s.ws_cap, (size_t)ws_stride * batch * s.S)) return rc;
  }
  const K4Grid* kg = static_cast<const K4Grid*>(s.d_grid);
  const K4Species* ks = static_cast<const K4Species*>(s.d_spec);
  if (s.warp_wpc && s.use_warp) {
    const int groups = (batch + s.warp_wpc - 1) / s.warp_wpc;
    k4_tfqmr_t<true><<<s.S * groups, 32 * s.warp_wpc, s.warp_smem, st>>>(kg, ks, s.S, batch, vals, s.v_stride, rhs, s.f_stride, x, rtol,
                                                                      max_it, iters, relres, nullptr, 0, s.warp_n, s.warp_nnz);
  } else {
    // small systems: fewer threads per system, several systems per SM (the iteration is latency bound)
    const int threads = s.max_n <= 256 ? 128 : s.max_n <= 1024 ? 256 : K4_THREADS;
    k4_tfqmr_t<false><<<batch * s.S, threads, s.smem, st>>>(kg, ks, s.S, batch, vals, s.v_stride, rhs, s.f_stride, x, rtol, max_it, iters,
                                                           relres, s.ws, ws_stride, s.mat_nnz ? ((s.max_n + 1) & ~1) : s.smem_n,
                                                           s.mat_nnz);
  }
  ++s.launches;
  SOLVER_TRY(s, cudaGetLastError());
  return LANDAU_OK;
}

// ------------------------------------------------------------------------------------------------------------
// landau_solve_noalloc: the Krylov workspace nobody allocates.
//
// Some users of this library cannot let it call cudaMalloc: their application owns all of the card's memory through a
// pool of its own, or runs a time-step loop in which the device-wide synchronisation of cudaMalloc / cudaFree is not
// acceptable.  For them the workspace of the large-system branch of k4_tfqmr (seven vectors per system in global memory)
// is this array, which is part of the loaded library image on every device from module load to process exit.
//
// On the HOST side `k4_noalloc_ws` is only a handle the runtime knows the symbol by -- it is not an address on any
// device, and a kernel handed `k4_noalloc_ws` from host code would read and write somewhere else entirely.  The address
// each device gave to its copy has to be asked for (cudaGetSymbolAddress) with that device current; noalloc_ws_address
// does so once per device and keeps the answer.
// ------------------------------------------------------------------------------------------------------------
constexpr unsigned long long K4_NOALLOC_WS_DOUBLES = LANDAU_SOLVE_NOALLOC_WS_BYTES / sizeof(double);
static __device__ __align__(256) double k4_noalloc_ws[K4_NOALLOC_WS_DOUBLES];

namespace {
std::mutex g_noalloc_mutex;
double* g_noalloc_addr[64] = {nullptr};  // per device ordinal: device address of that device's k4_noalloc_ws

int noalloc_ws_address(BatchSolver& s, double** out) {
  int dev = -1;
  SOLVER_TRY(s, cudaGetDevice(&dev));
  if (dev != s.device || dev < 0 || dev >= 64) {
    s.err = "landau_solve_noalloc: the context's device (ordinal < 64) must be the current device";
    return LANDAU_CUDA_ERROR;
  }
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  if (!g_noalloc_addr[dev]) {
    double* p = nullptr;
    SOLVER_TRY(s, cudaGetSymbolAddress(reinterpret_cast<void**>(&p), k4_noalloc_ws));
    if (!p) {
      s.err = "landau_solve_noalloc: cudaGetSymbolAddress returned a null address for the static workspace";
      return LANDAU_CUDA_ERROR;
    }
    g_noalloc_addr[dev] = p;
  }
  *out = g_noalloc_addr[dev];
  return LANDAU_OK;
}
}  // namespace

int solver_tfqmr_noalloc(BatchSolver& s, const double* vals, const double* rhs, int batch, double rtol, int max_it, double* x,
                         int* iters, double* relres, cudaStream_t st) {
  // the set-up of the first call on this device; later calls read the cached address
  double* ws = nullptr;
  if (int rc = noalloc_ws_address(s, &ws)) return rc;
  long long ws_stride = 0;
  if (s.max_n > s.smem_n) {  // same rule as solver_tfqmr: some grid's vectors do not fit in shared memory
    ws_stride = (long long)K4_NVEC * s.max_n;
    const unsigned long long need = (unsigned long long)ws_stride * (unsigned long long)batch * (unsigned long long)s.S;
    if (need > K4_NOALLOC_WS_DOUBLES) {
      const unsigned long long per_entry = (unsigned long long)ws_stride * (unsigned long long)s.S;
      s.err = "landau_solve_noalloc: " + std::to_string(batch) + " entries x " + std::to_string(s.S) + " species x 7 x " +
              std::to_string(s.max_n) + " unknowns = " + std::to_string(need * sizeof(double)) +
              " bytes of Krylov workspace, the static array holds LANDAU_SOLVE_NOALLOC_WS_BYTES = " +
              std::to_string(K4_NOALLOC_WS_DOUBLES * sizeof(double)) + ": at most batch = " +
              std::to_string(K4_NOALLOC_WS_DOUBLES / per_entry) + " per call on this context (split the batch, or use landau_solve)";
      return LANDAU_INVALID_ARG;
    }
  } else {
    ws = nullptr;  // every system keeps its vectors in shared memory: the array is not touched
  }
  // Nothing is cleared: k4_tfqmr writes idg, then rs / w / u / d, then au / v before the first read of each, so the
  // vectors a previous call left in the array are never seen.
  const int threads = s.max_n <= 256 ? 128 : s.max_n <= 1024 ? 256 : K4_THREADS;
  k4_tfqmr_t<false><<<batch * s.S, threads, s.smem, st>>>(static_cast<const K4Grid*>(s.d_grid), static_cast<const K4Species*>(s.d_spec),
                                                         s.S, batch, vals, s.v_stride, rhs, s.f_stride, x, rtol, max_it, iters,
                                                         relres, ws, ws_stride, s.mat_nnz ? ((s.max_n + 1) & ~1) : s.smem_n,
                                                         s.mat_nnz);
  ++s.launches;
  SOLVER_TRY(s, cudaGetLastError());
  return LANDAU_OK;
}

int solver_step(BatchSolver& s, const JacobianApplyFn& jacobian_apply, const double* mass_vals, double* u, int batch, double dt,
                double newton_rtol, int max_newton, double lin_rtol, int lin_max_it, double* info_host, cudaStream_t st) {
  s.err.clear();
  const size_t nf = (size_t)batch * s.f_stride, nsys = (size_t)batch * s.S;
  if (int rc = grow(s, &s.A, &s.A_cap, (size_t)batch * s.v_stride)) return rc;
  if (int rc = grow(s, &s.vec, &s.vec_cap, 4 * nf)) return rc;
  if (int rc = grow(s, &s.misc, &s.misc_cap, nsys + 2)) return rc;  // iteration counts (int) + scalar
  double *u0 = s.vec, *ju = u0 + nf, *rhs = ju + nf, *delta = rhs + nf;
  int* iters = reinterpret_cast<int*>(s.misc);
  unsigned long long* max_rel = reinterpret_cast<unsigned long long*>(s.misc + (nsys + 1) / 2 + 1);
  const K4Grid* kg = static_cast<const K4Grid*>(s.d_grid);
  const K4Species* ks = static_cast<const K4Species*>(s.d_spec);
  SOLVER_TRY(s, cudaMemcpyAsync(u0, u, sizeof(double) * nf, cudaMemcpyDeviceToDevice, st));
  const int eb = (int)std::min<size_t>((nf + 255) / 256, 65535);
  int it = 0, worst_lin = 0, lin_failed = 0, last_failed = 0;
  double rel = 0.0;
  std::vector<int> h_iters(nsys);
  for (it = 0; it < max_newton; ++it) {
    // A = M/dt - J[u], ju = J[u] u from one inner integral
    if (int rc = jacobian_apply(u, batch, dt, s.A, ju)) return rc;
    // rhs = M (u0 - u)/dt + J[u] u
    k5_axpby<<<eb, 256, 0, st>>>((long long)nf, 1.0, u0, -1.0, u, delta);
    k4_spmv_batch<<<batch * s.S, K4_THREADS, 0, st>>>(kg, ks, s.S, mass_vals, 0, delta, s.f_stride, rhs);
    k5_axpby<<<eb, 256, 0, st>>>((long long)nf, 1.0 / dt, rhs, 1.0, ju, rhs);
    s.launches += 3;
    SOLVER_TRY(s, cudaMemsetAsync(delta, 0, sizeof(double) * nf, st));
    if (int rc = solver_tfqmr(s, s.A, rhs, batch, lin_rtol, lin_max_it, delta, iters, nullptr, st)) return rc;
    SOLVER_TRY(s, cudaMemsetAsync(max_rel, 0, sizeof(unsigned long long), st));
    k5_update<<<batch * s.S, 256, 0, st>>>(kg, ks, s.S, u, delta, s.f_stride, max_rel);
    ++s.launches;
    unsigned long long bits = 0;
    SOLVER_TRY(s, cudaMemcpyAsync(&bits, max_rel, sizeof(bits), cudaMemcpyDeviceToHost, st));
    SOLVER_TRY(s, cudaMemcpyAsync(h_iters.data(), iters, sizeof(int) * nsys, cudaMemcpyDeviceToHost, st));
    SOLVER_TRY(s, cudaStreamSynchronize(st));
    memcpy(&rel, &bits, sizeof(rel));
    last_failed = 0;
    for (int v : h_iters) {
      worst_lin = std::max(worst_lin, v < 0 ? -v - 1 : v);
      last_failed += v < 0;
    }
    lin_failed += last_failed;
    if (rel <= newton_rtol) {
      ++it;
      break;
    }
  }
  if (info_host) {
    info_host[0] = it;
    info_host[1] = rel;
    info_host[2] = worst_lin;
    info_host[3] = lin_failed;
  }
  // u holds the last iterate either way; a caller without info_host must still learn that it is not the step's solution
  if (rel > newton_rtol || last_failed > 0) {
    s.err = "step not converged: largest relative update " + std::to_string(rel) + " after " + std::to_string(it) +
            " Newton iterations (newton_rtol " + std::to_string(newton_rtol) + "), " + std::to_string(last_failed) +
            " linear solves of the last iteration missed lin_rtol";
    return LANDAU_NOT_CONVERGED;
  }
  return LANDAU_OK;
}

}  // namespace landau
