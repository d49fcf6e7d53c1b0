// k4_solve.cuh -- batched linear solve of the shifted systems the Jacobian construction produces:
//
//     (M/dt - J[f]) x = b      one system per (batch entry, species)
//
// TFQMR (Freund; Saad Alg. 7.8) with left Jacobi preconditioning, the whole iteration of one system in ONE CTA, one
// launch for the batch (the paper's batched solver: "the entire solve requires a single kernel launch,
// each solve can run asynchronously, exiting the kernel as soon as it converges").  The seven Krylov vectors of a
// system live in shared memory (7 n doubles: 205 KB for the 3655 unknowns of the 14 x 28 Q3 grid, one CTA per SM), x
// in global memory; the CSR values of the systems in flight (148 x 0.7 MB) stay L2-resident over the iterations, the
// pattern (rowptr / colidx / diagonal positions) is shared by all systems of a grid.  SpMV: 8 lanes per row (24 nonzeros
// per row on Q3 grids), rows contiguous in the value array.  Systems whose vectors do not fit in shared memory take
// the same code with the vectors in a global workspace.
#pragma once

namespace landau {

struct K4Grid {
  int n, nnz;
  const int *rowptr, *colidx, *diag;  // diag[i] = position of a_ii in the row-major value array
};

struct K4Species {
  int grid;
  long long f_off, v_off;
};

constexpr int K4_THREADS = 512;  // largest CTA; small systems run with 128 or 256 threads (several CTAs per SM)
constexpr int K4_NVEC = 7;
constexpr int K4_RUN_CAP = 600;  // half-steps of one TFQMR run before it is restarted from the current x

// sums of two values over the CTA (deterministic order), result in every thread
__device__ __forceinline__ void k4_block_sum2(double& a, double& b, double* red) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    a += __shfl_xor_sync(0xffffffffu, a, o);
    b += __shfl_xor_sync(0xffffffffu, b, o);
  }
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  __syncthreads();  // red may still be read from the previous reduction
  if (lane == 0) {
    red[2 * warp] = a;
    red[2 * warp + 1] = b;
  }
  __syncthreads();
  a = 0.0;
  b = 0.0;
  const int nw = blockDim.x >> 5;
  for (int wv = 0; wv < nw; ++wv) {
    a += red[2 * wv];
    b += red[2 * wv + 1];
  }
}

// out(row, sum_k a_ik in_k) for every row: 8 lanes per row, two rows per lane group in flight, the first 48 entries of
// a row loaded into registers before the first use (values and indices come from L2: memory-level parallelism is what
// counts), longer rows (hanging-node rows) finish in a tail loop.
constexpr int K4_T = 6;  // entries per lane held in registers per row (8 lanes: rows up to 48 entries without a tail)

template <bool LDG, class T>
__device__ __forceinline__ T k4_ld(const T* p) {
  if constexpr (LDG)
    return __ldg(p);
  else
    return *p;
}

// LDG: pattern and values in global memory (read-only path); otherwise they may sit in shared memory (plain loads)
// tid / nthreads: the thread's index in, and the size of, the group that owns the system (the CTA, or one warp of it)
template <bool LDG = true, class Out>
__device__ __forceinline__ void k4_spmv(const K4Grid& g, const double* __restrict__ vals, const double* in, Out out,
                                        int tid = threadIdx.x, int nthreads = blockDim.x) {
  const int l8 = tid & 7, sub = (tid & 31) >> 3;
  const int RS = nthreads >> 3;  // rows per sweep of the group
  constexpr int U = 2;                // rows per lane group in flight
  // warp-uniform trip count (the shuffles need all 32 lanes; rows past the end contribute nothing); the row bounds of
  // the next iteration are fetched while the current rows are summed.  All value / index loads of an iteration are
  // issued before the first use: the product is bound by the latency of those loads (L2), not by their volume.
  int k0[U], k1[U];
  const int first = (tid >> 5) * 4;
  auto bounds = [&](int row0) {
#pragma unroll
    for (int j = 0; j < U; ++j) {
      const int r = row0 + j * RS + sub;
      const bool live = r < g.n;
      k0[j] = live ? k4_ld<LDG>(g.rowptr + r) : 0;
      k1[j] = live ? k4_ld<LDG>(g.rowptr + r + 1) : 0;
    }
  };
  bounds(first);
  for (int row0 = first; row0 < g.n; row0 += U * RS) {
    double av[U][K4_T];
    int ci[U][K4_T], c0[U], c1[U];
#pragma unroll
    for (int j = 0; j < U; ++j) {
      c0[j] = k0[j];
      c1[j] = k1[j];
#pragma unroll
      for (int t = 0; t < K4_T; ++t) {
        const int k = c0[j] + l8 + 8 * t;
        const bool p = k < c1[j];
        av[j][t] = p ? k4_ld<LDG>(vals + k) : 0.0;
        ci[j][t] = p ? k4_ld<LDG>(g.colidx + k) : 0;
      }
    }
    if (row0 + U * RS < g.n) bounds(row0 + U * RS);
    double sum[U];
#pragma unroll
    for (int j = 0; j < U; ++j) {
      double sj = 0.0;
#pragma unroll
      for (int t = 0; t < K4_T; ++t) sj = fma(av[j][t], in[ci[j][t]], sj);
      for (int k = c0[j] + l8 + 8 * K4_T; k < c1[j]; k += 8) sj = fma(k4_ld<LDG>(vals + k), in[k4_ld<LDG>(g.colidx + k)], sj);
      sum[j] = sj;
    }
#pragma unroll
    for (int o = 4; o > 0; o >>= 1)
#pragma unroll
      for (int j = 0; j < U; ++j) sum[j] += __shfl_xor_sync(0xffffffffu, sum[j], o);
    if (l8 == 0) {
#pragma unroll
      for (int j = 0; j < U; ++j) {
        const int r = row0 + j * RS + sub;
        if (r < g.n) out(r, sum[j]);
      }
    }
  }
}

// sums of two values over one warp, result in every lane
__device__ __forceinline__ void k4_warp_sum2(double& a, double& b) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    a += __shfl_xor_sync(0xffffffffu, a, o);
    b += __shfl_xor_sync(0xffffffffu, b, o);
  }
}

// WARP = false: one system per CTA (blockIdx.x = entry * n_spec + species).
// WARP = true (small systems): one system per WARP, no block-wide barrier anywhere in the iteration -- a CTA of `wpc` warps
// takes wpc entries of ONE species (blockIdx.x = species * ceil(batch / wpc) + entry group), so that its warps share the
// pattern of that species' grid in shared memory; every warp keeps its own values and vectors there.
template <bool WARP>
__global__ void __launch_bounds__(K4_THREADS)
k4_tfqmr_t(const K4Grid* __restrict__ grids, const K4Species* __restrict__ spec, int n_spec, int batch,
           const double* __restrict__ vals, long long v_stride, const double* __restrict__ rhs, long long f_stride,
           double* __restrict__ x, double rtol, int max_it, int* __restrict__ iters, double* __restrict__ relres,
           double* __restrict__ ws, long long ws_stride, int smem_n, int mat_nnz) {
  extern __shared__ __align__(16) double k4_smem[];
  double* red = k4_smem;  // [2 * warps]
  const int wpc = blockDim.x >> 5, warp = threadIdx.x >> 5;
  int sidx, b;
  if (WARP) {
    const int groups = (batch + wpc - 1) / wpc;
    sidx = blockIdx.x / groups;
    b = (blockIdx.x - sidx * groups) * wpc + warp;
  } else {
    sidx = blockIdx.x % n_spec;
    b = blockIdx.x / n_spec;
  }
  const int sys = b * n_spec + sidx;  // index of the system in iters / relres / ws
  const K4Species sp = spec[sidx];
  K4Grid g = grids[sp.grid];
  const int n = g.n, tid = WARP ? (int)(threadIdx.x & 31) : (int)threadIdx.x, nthreads = WARP ? 32 : (int)blockDim.x;
  auto sync = [&]() {
    if (WARP)
      __syncwarp();
    else
      __syncthreads();
  };
  auto sum2 = [&](double& p, double& q) {
    if (WARP)
      k4_warp_sum2(p, q);
    else
      k4_block_sum2(p, q, red);
  };
  // shared memory, WARP: [pattern of the grid: colidx (mat_nnz ints), rowptr (smem_n + 2 ints)] then per warp
  // [7 vectors of smem_n doubles | mat_nnz values];  otherwise: [red | 7 vectors | values | colidx | rowptr]
  double* vec;
  if (WARP) {
    int* scol = reinterpret_cast<int*>(k4_smem);
    int* srow = scol + mat_nnz;
    for (int k = threadIdx.x; k < g.nnz; k += blockDim.x) scol[k] = g.colidx[k];
    for (int i = threadIdx.x; i <= n; i += blockDim.x) srow[i] = g.rowptr[i];
    g.colidx = scol;
    g.rowptr = srow;
    double* base = k4_smem + ((mat_nnz + smem_n + 2 + 1) >> 1);
    vec = base + (long long)warp * ((long long)K4_NVEC * smem_n + mat_nnz);
    __syncthreads();  // the only block-wide barrier: the shared pattern is in place
    if (b >= batch) return;
  } else {
    vec = n <= smem_n ? k4_smem + 2 * (K4_THREADS / 32) : ws + (long long)sys * ws_stride;
  }
  double *rs = vec, *w = vec + n, *u = vec + 2 * n, *v = vec + 3 * n, *d = vec + 4 * n, *au = vec + 5 * n, *idg = vec + 6 * n;
  const double* a = vals + (long long)b * v_stride + sp.v_off;  // re-pointed to shared memory for small systems
  const double* bb = rhs + (long long)b * f_stride + sp.f_off;
  double* xx = x + (long long)b * f_stride + sp.f_off;

  for (int i = tid; i < n; i += nthreads) idg[i] = 1.0 / a[g.diag[i]];
  // Small systems (mat_nnz > 0: every grid's pattern and one value block fit beside the vectors): the matrix is copied
  // to shared memory once, and the products of the iteration run from there instead of from L2.
  const bool mat_smem = mat_nnz > 0;
  if (WARP) {
    double* sval = vec + (long long)K4_NVEC * smem_n;
    for (int k = tid; k < g.nnz; k += 32) sval[k] = a[k];
    a = sval;
  } else if (mat_smem) {
    double* sval = k4_smem + 2 * (K4_THREADS / 32) + (long long)K4_NVEC * smem_n;
    int* scol = reinterpret_cast<int*>(sval + mat_nnz);
    int* srow = scol + mat_nnz;
    for (int k = tid; k < g.nnz; k += nthreads) {
      sval[k] = a[k];
      scol[k] = g.colidx[k];
    }
    for (int i = tid; i <= n; i += nthreads) srow[i] = g.rowptr[i];
    a = sval;
    g.colidx = scol;
    g.rowptr = srow;
  }
  sync();
  auto product = [&](const double* in, auto out) {
    if (WARP || mat_smem)
      k4_spmv<false>(g, a, in, out, tid, nthreads);
    else
      k4_spmv<true>(g, a, in, out, tid, nthreads);
  };
  // TFQMR's residual bound is updated recursively and drifts away from the true residual on ill-conditioned blocks,
  // so a converged run is CHECKED against the true (Jacobi-scaled) residual and restarted from the current x if it
  // misses the tolerance, which stays relative to the first residual.  A run is also restarted after K4_RUN_CAP
  // half-steps: with the shadow residual fixed, TFQMR can stagnate for thousands of steps on the electron blocks of
  // the large grids (cond(D^-1 A) ~ 5e3), and a restart from the current iterate ends that.
  double r0norm = 0.0, tau = 0.0;
  int m = 0, status = 0;  // 1 converged, 2 breakdown, 0 running / not converged
  for (int restart = 0; !status; ++restart) {
    // r = D^-1 (b - A x);  w = u = rs = r, d = 0
    product(xx, [&](int row, double s) {
      const double r = idg[row] * (bb[row] - s);
      rs[row] = r;
      w[row] = r;
      u[row] = r;
      d[row] = 0.0;
    });
    sync();
    double p0 = 0.0, p1 = 0.0;
    for (int i = tid; i < n; i += nthreads) p0 = fma(rs[i], rs[i], p0);
    sum2(p0, p1);
    double rho = p0, theta = 0.0, eta = 0.0, alpha = 0.0;
    tau = sqrt(p0);
    if (restart == 0) r0norm = tau;
    if (tau <= rtol * r0norm) {  // true residual within tolerance (also: zero right-hand side)
      status = 1;
      break;
    }
    if (m >= 2 * max_it) break;
    product(u, [&](int row, double s) {
      const double t = idg[row] * s;
      au[row] = t;
      v[row] = t;
    });
    sync();
    bool bound_met = false;
    for (int k = 0; !bound_met && !status && m < 2 * max_it && k < K4_RUN_CAP; ++k) {  // k: half-step of this run
      const bool even = (k & 1) == 0;
      if (even) {
        double sg = 0.0, z = 0.0;
        for (int i = tid; i < n; i += nthreads) sg = fma(rs[i], v[i], sg);
        sum2(sg, z);
        if (sg == 0.0) {
          status = 2;
          break;
        }
        alpha = rho / sg;
      }
      // w -= alpha A u;  d = u + (theta^2 eta / alpha) d;  ||w||^2 and (rs, w)
      const double cd = theta * theta * eta / alpha;
      double ww = 0.0, rw = 0.0;
      for (int i = tid; i < n; i += nthreads) {
        const double wi = fma(-alpha, au[i], w[i]);
        w[i] = wi;
        d[i] = fma(cd, d[i], u[i]);
        ww = fma(wi, wi, ww);
        rw = fma(rs[i], wi, rw);
      }
      sum2(ww, rw);
      theta = sqrt(ww) / tau;
      const double c = 1.0 / sqrt(1.0 + theta * theta);
      tau = tau * theta * c;
      eta = c * c * alpha;
      for (int i = tid; i < n; i += nthreads) xx[i] = fma(eta, d[i], xx[i]);
      ++m;
      if (tau * sqrt((double)(k + 1)) <= rtol * r0norm) {
        bound_met = true;
      } else if (even) {
        for (int i = tid; i < n; i += nthreads) u[i] = fma(-alpha, v[i], u[i]);
        sync();
        product(u, [&](int row, double s) { au[row] = idg[row] * s; });
      } else {
        if (rho == 0.0) {
          status = 2;
          break;
        }
        const double beta = rw / rho;
        rho = rw;
        for (int i = tid; i < n; i += nthreads) u[i] = fma(beta, u[i], w[i]);
        sync();
        // v = A u_new + beta (A u_old + beta v);  au = A u_new
        product(u, [&](int row, double s) {
          const double t = idg[row] * s;
          v[row] = fma(beta, fma(beta, v[row], au[row]), t);
          au[row] = t;
        });
      }
      sync();
    }
    if (status == 2) break;  // breakdown
    // bound met: verify against the true residual; run cap reached: restart (a fresh shadow residual ends stagnation)
  }
  if (tid == 0) {
    if (iters) iters[sys] = status == 1 ? m : -m - 1;  // half-steps; negative: not converged / breakdown
    if (relres) relres[sys] = r0norm > 0.0 ? tau / r0norm : 0.0;  // last true residual seen (or bound)
  }
}

// y = A x for every (entry, species) block (residual checks, right-hand sides M f / dt)
__global__ void __launch_bounds__(K4_THREADS)
k4_spmv_batch(const K4Grid* __restrict__ grids, const K4Species* __restrict__ spec, int n_spec,
              const double* __restrict__ vals, long long v_stride, const double* __restrict__ x, long long f_stride,
              double* __restrict__ y) {
  const int sidx = blockIdx.x % n_spec, b = blockIdx.x / n_spec;
  const K4Species sp = spec[sidx];
  const K4Grid g = grids[sp.grid];
  double* yy = y + (long long)b * f_stride + sp.f_off;
  k4_spmv(g, vals + (long long)b * v_stride + sp.v_off, x + (long long)b * f_stride + sp.f_off,
          [&](int row, double s) { yy[row] = s; });
}

// ------------------------------------------------------------------------------------------------------------
// Small kernels of the backward-Euler quasi-Newton step (landau_step): out = a x + b y, and the update u += delta with
// the largest relative update over the (entry, species) blocks (positive doubles order like their bit patterns).
// ------------------------------------------------------------------------------------------------------------
__global__ void k5_axpby(long long n, double a, const double* __restrict__ x, double b, const double* __restrict__ y,
                         double* __restrict__ out) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
    out[i] = a * x[i] + b * y[i];
}

__global__ void __launch_bounds__(256)
k5_update(const K4Grid* __restrict__ grids, const K4Species* __restrict__ spec, int n_spec, double* __restrict__ u,
          const double* __restrict__ delta, long long f_stride, unsigned long long* __restrict__ max_rel_bits) {
  __shared__ double red[2 * 8];
  const int sidx = blockIdx.x % n_spec, b = blockIdx.x / n_spec;
  const K4Species sp = spec[sidx];
  const int n = grids[sp.grid].n;
  double* uu = u + (long long)b * f_stride + sp.f_off;
  const double* dd = delta + (long long)b * f_stride + sp.f_off;
  double d2 = 0.0, u2 = 0.0;
  for (int i = threadIdx.x; i < n; i += 256) {
    const double di = dd[i], ui = uu[i] + di;
    uu[i] = ui;
    d2 = fma(di, di, d2);
    u2 = fma(ui, ui, u2);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    d2 += __shfl_xor_sync(0xffffffffu, d2, o);
    u2 += __shfl_xor_sync(0xffffffffu, u2, o);
  }
  if ((threadIdx.x & 31) == 0) {
    red[2 * (threadIdx.x >> 5)] = d2;
    red[2 * (threadIdx.x >> 5) + 1] = u2;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    d2 = u2 = 0.0;
    for (int w = 0; w < 8; ++w) {
      d2 += red[2 * w];
      u2 += red[2 * w + 1];
    }
    const double rel = u2 > 0.0 ? sqrt(d2 / u2) : 0.0;
    atomicMax(max_rel_bits, (unsigned long long)__double_as_longlong(rel));
  }
}

}  // namespace landau
