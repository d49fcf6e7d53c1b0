// landau3v_kernels.cuh -- device kernels of the 3V variant (include/landau3v.h).
//
//   K1  k3v_fields        a1: w_j {f, grad f} of every source column at the integration points
//   K2  k3v_inner_dfma    a2: G^D (6) and G^K (3) of every column at every integration point, scalar FP64 pipe
//       k3v_inner_dmma    a2: the same contraction on the FP64 MMA (m8n8k4), tensor generated per warp
//   K2b k3v_combine       a2: D_a, K_a = species combination of the G's
//   K3  k3v_assemble      a3 + a4: element-matrix entries by quadrature, gathered per CSR slot, written once
//   K3' k3v_elem_apply, k3v_apply_gather   a5
//
// Source columns: with a rank-one nu (nu_ab = a_a b_b) the species sum is folded into the source field, one column
// per batch entry over the points of ALL grids; otherwise one column per (entry, species) that is non-zero on that
// species' grid only.  F is stored [class][entry][4][n_pad] (class = 0 or the species), G [class][entry][9][n_pad].
#pragma once
#include <cuda_runtime.h>

namespace landau3v {

constexpr int K2_TJ = 64;      // source points per shared-memory tile
constexpr int K2_TI = 128;     // field points per CTA of the scalar kernel (one per thread)
constexpr int MAX_TERMS = 16;  // species (general nu) / species per grid (mix)

struct DevGrid3 {
  int n_cells, n_dof, n_ip, nnz, ip_off;
  const double *cell_h, *ip_w;
  const int *en_ptr, *en_dof;
  const double* en_w;
  const int *as_ptr, *as_code;
  const double* as_w;
  const int *ap_ptr, *ap_code;
  const double* ap_w;
};

struct Tables3 {
  double B[729], dBx[729], dBy[729], dBz[729];  // [q][a]
};

// which species of a grid go into which column class, with which weights (D part: f, K part: grad f)
struct Mix3 {
  int n_entries;
  int cls[MAX_TERMS], f_off[MAX_TERMS];
  double wD[MAX_TERMS], wK[MAX_TERMS];
};

// D_a = sum_t coefD[t] G^D[class cls[t]],  K_a likewise
struct Combine3 {
  int n_terms, ip_off, n_ip;
  long long dk_off;
  int cls[MAX_TERMS];
  double coefD[MAX_TERMS], coefK[MAX_TERMS];
};

// ---------------------------------------------------------------------------------------------------------------- K1
// grid (n_cells, nbc), 32 threads: thread a < 27 expands nodal value a through the constraints, thread q < 27 contracts
__global__ void __launch_bounds__(32) k3v_fields(DevGrid3 g, const Tables3* __restrict__ tab, Mix3 mix,
                                                const double* __restrict__ batch_f, long long f_stride, int b0, int nbc,
                                                double* __restrict__ F, int n_pad) {
  __shared__ double nd[27], nk[27];
  const int cell = blockIdx.x, b = blockIdx.y, t = threadIdx.x;
  const double* f = batch_f + (long long)(b0 + b) * f_stride;
  const double sc = 2.0 / g.cell_h[cell];
  for (int m0 = 0; m0 < mix.n_entries;) {
    const int cls = mix.cls[m0];
    int m1 = m0;
    while (m1 < mix.n_entries && mix.cls[m1] == cls) ++m1;
    if (t < 27) {
      double vd = 0.0, vk = 0.0;
      for (int p = g.en_ptr[cell * 27 + t]; p < g.en_ptr[cell * 27 + t + 1]; ++p) {
        const double w = g.en_w[p];
        const int dof = g.en_dof[p];
        for (int m = m0; m < m1; ++m) {
          const double v = w * f[mix.f_off[m] + dof];
          vd = fma(mix.wD[m], v, vd);
          vk = fma(mix.wK[m], v, vk);
        }
      }
      nd[t] = vd;
      nk[t] = vk;
    }
    __syncwarp();
    if (t < 27) {
      double v = 0.0, gx = 0.0, gy = 0.0, gz = 0.0;
#pragma unroll 9
      for (int a = 0; a < 27; ++a) {
        v = fma(tab->B[t * 27 + a], nd[a], v);
        gx = fma(tab->dBx[t * 27 + a], nk[a], gx);
        gy = fma(tab->dBy[t * 27 + a], nk[a], gy);
        gz = fma(tab->dBz[t * 27 + a], nk[a], gz);
      }
      const int ip = cell * 27 + t;
      const double w = g.ip_w[ip], ws = w * sc;
      double* dst = F + ((long long)cls * nbc + b) * 4 * n_pad + g.ip_off + ip;
      dst[0] = w * v;
      dst[n_pad] = ws * gx;
      dst[2 * (long long)n_pad] = ws * gy;
      dst[3 * (long long)n_pad] = ws * gz;
    }
    __syncwarp();
    m0 = m1;
  }
}

// ---------------------------------------------------------------------------------------------------------------- K2
// The Landau tensor of one pair: U = (|u|^2 I - u u^T) / |u|^3; zero for coincident points.
struct Tensor6 {
  double xx, xy, xz, yy, yz, zz;
};
__device__ __forceinline__ Tensor6 landau_tensor_3v(double xi, double yi, double zi, double ri2, double xj, double yj,
                                                    double zj) {
  const double ux = xi - xj, uy = yi - yj, uz = zi - zj;
  const double u2 = fma(ux, ux, fma(uy, uy, uz * uz));
  const double scale = ri2 + fma(xj, xj, fma(yj, yj, zj * zj));
  double inv = rsqrt(u2);
  inv = u2 > 1e-20 * scale ? inv : 0.0;
  const double inv3 = inv * inv * inv;
  Tensor6 U;
  U.xx = (u2 - ux * ux) * inv3;
  U.yy = (u2 - uy * uy) * inv3;
  U.zz = (u2 - uz * uz) * inv3;
  const double m = -inv3;
  U.xy = ux * uy * m;
  U.xz = ux * uz * m;
  U.yz = uy * uz * m;
  return U;
}

// grid (n_pad / 128, tiles), 128 threads: thread = field point, NC columns of one class, source tiles in shared memory.
// class c reads the source range [j0[c], j1[c]) (multiples of K2_TJ; F of the class is zero outside its own grid).
struct Ranges3 {
  int j0[MAX_TERMS], j1[MAX_TERMS];
};
template <int NC>
__global__ void __launch_bounds__(K2_TI) k3v_inner_dfma(const double* __restrict__ px, const double* __restrict__ py,
                                                        const double* __restrict__ pz, int n_pad, Ranges3 rg, int nbc,
                                                        const double* __restrict__ F, double* __restrict__ G) {
  __shared__ double sx[K2_TJ], sy[K2_TJ], sz[K2_TJ], sF[NC][4][K2_TJ];
  const int tiles_per_class = (nbc + NC - 1) / NC;
  const int cls = blockIdx.y / tiles_per_class, bfirst = (blockIdx.y % tiles_per_class) * NC;
  const int i = blockIdx.x * K2_TI + threadIdx.x;
  const double xi = px[i], yi = py[i], zi = pz[i];
  const double ri2 = fma(xi, xi, fma(yi, yi, zi * zi));
  double acc[NC][9];
#pragma unroll
  for (int n = 0; n < NC; ++n)
#pragma unroll
    for (int k = 0; k < 9; ++k) acc[n][k] = 0.0;
  const double* Fc = F + ((long long)cls * nbc + bfirst) * 4 * n_pad;
  for (int jt = rg.j0[cls]; jt < rg.j1[cls]; jt += K2_TJ) {
    __syncthreads();
    if (threadIdx.x < K2_TJ) {
      sx[threadIdx.x] = px[jt + threadIdx.x];
      sy[threadIdx.x] = py[jt + threadIdx.x];
      sz[threadIdx.x] = pz[jt + threadIdx.x];
    }
    for (int e = threadIdx.x; e < NC * 4 * K2_TJ; e += K2_TI) {
      const int n = e / (4 * K2_TJ), r = e % (4 * K2_TJ);
      sF[n][r / K2_TJ][r % K2_TJ] = bfirst + n < nbc ? Fc[((long long)n * 4 + r / K2_TJ) * n_pad + jt + r % K2_TJ] : 0.0;
    }
    __syncthreads();
#pragma unroll 2
    for (int j = 0; j < K2_TJ; ++j) {
      const Tensor6 U = landau_tensor_3v(xi, yi, zi, ri2, sx[j], sy[j], sz[j]);
#pragma unroll
      for (int n = 0; n < NC; ++n) {
        const double f = sF[n][0][j], gx = sF[n][1][j], gy = sF[n][2][j], gz = sF[n][3][j];
        acc[n][0] = fma(U.xx, f, acc[n][0]);
        acc[n][1] = fma(U.xy, f, acc[n][1]);
        acc[n][2] = fma(U.xz, f, acc[n][2]);
        acc[n][3] = fma(U.yy, f, acc[n][3]);
        acc[n][4] = fma(U.yz, f, acc[n][4]);
        acc[n][5] = fma(U.zz, f, acc[n][5]);
        acc[n][6] = fma(U.xx, gx, fma(U.xy, gy, fma(U.xz, gz, acc[n][6])));
        acc[n][7] = fma(U.xy, gx, fma(U.yy, gy, fma(U.yz, gz, acc[n][7])));
        acc[n][8] = fma(U.xz, gx, fma(U.yz, gy, fma(U.zz, gz, acc[n][8])));
      }
    }
  }
#pragma unroll
  for (int n = 0; n < NC; ++n)
    if (bfirst + n < nbc) {
      double* dst = G + ((long long)cls * nbc + bfirst + n) * 9 * n_pad + i;
#pragma unroll
      for (int k = 0; k < 9; ++k) dst[(long long)k * n_pad] = acc[n][k];
    }
}

// --------------------------------------------------------------------------------------------------------------- K2b
// grid (ceil(max n_ip / 256), nbc, S); the `nsplit` partial sums of a cut source range are added here, in part order
__global__ void __launch_bounds__(256) k3v_combine(const Combine3* __restrict__ comb, const double* __restrict__ G, int n_pad,
                                                   int nbc, int nsplit, long long split_stride, double* __restrict__ DK,
                                                   long long dk_stride) {
  const Combine3& c = comb[blockIdx.z];
  const int i = blockIdx.x * 256 + threadIdx.x, b = blockIdx.y;
  if (i >= c.n_ip) return;
  double out[9];
#pragma unroll
  for (int k = 0; k < 9; ++k) out[k] = 0.0;
  for (int t = 0; t < c.n_terms; ++t) {
    const double* src = G + ((long long)c.cls[t] * nbc + b) * 9 * n_pad + c.ip_off + i;
    const double cd = c.coefD[t], ck = c.coefK[t];
#pragma unroll
    for (int k = 0; k < 9; ++k) {
      double g = src[(long long)k * n_pad];
      for (int sp = 1; sp < nsplit; ++sp) g += src[sp * split_stride + (long long)k * n_pad];
      out[k] = fma(k < 6 ? cd : ck, g, out[k]);
    }
  }
  double* dst = DK + (long long)b * dk_stride + c.dk_off + i;
#pragma unroll
  for (int k = 0; k < 9; ++k) dst[(long long)k * c.n_ip] = out[k];
}

// ---------------------------------------------------------------------------------------------------------------- K3
// grid (ceil(nnz / 128), nbc), 128 threads: one thread per CSR slot; every contribution A_cell[a][c] is integrated on the
// fly,  A[a][c] = sum_q w_q [ phi_a phi_c / dt + grad phi_a . D grad phi_c - (grad phi_a . K) phi_c ].
// Threads of a warp hold neighbouring slots of a row, i.e. mostly the same cell: the D, K loads are broadcasts.
__global__ void __launch_bounds__(128) k3v_assemble(DevGrid3 g, const Tables3* __restrict__ tab, const double* __restrict__ DK,
                                                    long long dk_stride, long long dk_off, double inv_dt,
                                                    double* __restrict__ vals, long long v_stride, long long v_off) {
  __shared__ double sB[729], sX[729], sY[729], sZ[729];
  for (int e = threadIdx.x; e < 729; e += 128) {
    sB[e] = tab->B[e];
    sX[e] = tab->dBx[e];
    sY[e] = tab->dBy[e];
    sZ[e] = tab->dBz[e];
  }
  __syncthreads();
  const int n = blockIdx.x * 128 + threadIdx.x, b = blockIdx.y;
  if (n >= g.nnz) return;
  const double* dk = DK + (long long)b * dk_stride + dk_off;
  const long long N = g.n_ip;
  double v = 0.0;
  for (int p = g.as_ptr[n]; p < g.as_ptr[n + 1]; ++p) {
    const int code = g.as_code[p], c = code % 27, a = (code / 27) % 27, cell = code / 729;
    const double sc = 2.0 / g.cell_h[cell], sc2 = sc * sc;
    double acc = 0.0;
    for (int q = 0; q < 27; ++q) {
      const int ip = cell * 27 + q;
      const double w = g.ip_w[ip];
      const double ax = sX[q * 27 + a], ay = sY[q * 27 + a], az = sZ[q * 27 + a];
      const double cx = sX[q * 27 + c], cy = sY[q * 27 + c], cz = sZ[q * 27 + c];
      const double dxx = dk[ip], dxy = dk[N + ip], dxz = dk[2 * N + ip], dyy = dk[3 * N + ip], dyz = dk[4 * N + ip],
                   dzz = dk[5 * N + ip];
      const double kx = dk[6 * N + ip], ky = dk[7 * N + ip], kz = dk[8 * N + ip];
      const double dterm = ax * (dxx * cx + dxy * cy + dxz * cz) + ay * (dxy * cx + dyy * cy + dyz * cz) +
                           az * (dxz * cx + dyz * cy + dzz * cz);
      const double kterm = ax * kx + ay * ky + az * kz;
      const double pc = sB[q * 27 + c];
      acc = fma(w, fma(sc2, dterm, fma(inv_dt * sB[q * 27 + a], pc, -sc * kterm * pc)), acc);
    }
    v = fma(g.as_w[p], acc, v);
  }
  __stcs(vals + (long long)b * v_stride + v_off + n, v);
}

// --------------------------------------------------------------------------------------------------------------- K3'
// grid (n_cells, nbc), 32 threads: nodal values -> f, grad f -> weighted flux at the points -> element vector
__global__ void __launch_bounds__(32) k3v_elem_apply(DevGrid3 g, const Tables3* __restrict__ tab,
                                                    const double* __restrict__ batch_f, long long f_stride, long long f_off,
                                                    int b0, const double* __restrict__ DK, long long dk_stride,
                                                    long long dk_off, double* __restrict__ FE, long long fe_stride,
                                                    long long fe_off) {
  __shared__ double nd[27], fl[3][27];
  const int cell = blockIdx.x, b = blockIdx.y, t = threadIdx.x;
  const double* f = batch_f + (long long)(b0 + b) * f_stride + f_off;
  const double sc = 2.0 / g.cell_h[cell];
  if (t < 27) {
    double v = 0.0;
    for (int p = g.en_ptr[cell * 27 + t]; p < g.en_ptr[cell * 27 + t + 1]; ++p) v = fma(g.en_w[p], f[g.en_dof[p]], v);
    nd[t] = v;
  }
  __syncwarp();
  if (t < 27) {
    double v = 0.0, gx = 0.0, gy = 0.0, gz = 0.0;
    for (int a = 0; a < 27; ++a) {
      v = fma(tab->B[t * 27 + a], nd[a], v);
      gx = fma(tab->dBx[t * 27 + a], nd[a], gx);
      gy = fma(tab->dBy[t * 27 + a], nd[a], gy);
      gz = fma(tab->dBz[t * 27 + a], nd[a], gz);
    }
    gx *= sc;
    gy *= sc;
    gz *= sc;
    const long long N = g.n_ip;
    const int ip = cell * 27 + t;
    const double* dk = DK + (long long)b * dk_stride + dk_off + ip;
    const double w = g.ip_w[ip] * sc;
    fl[0][t] = w * (-(dk[0] * gx + dk[N] * gy + dk[2 * N] * gz) + dk[6 * N] * v);
    fl[1][t] = w * (-(dk[N] * gx + dk[3 * N] * gy + dk[4 * N] * gz) + dk[7 * N] * v);
    fl[2][t] = w * (-(dk[2 * N] * gx + dk[4 * N] * gy + dk[5 * N] * gz) + dk[8 * N] * v);
  }
  __syncwarp();
  if (t < 27) {
    double r = 0.0;
    for (int q = 0; q < 27; ++q)
      r = fma(tab->dBx[q * 27 + t], fl[0][q], fma(tab->dBy[q * 27 + t], fl[1][q], fma(tab->dBz[q * 27 + t], fl[2][q], r)));
    FE[(long long)b * fe_stride + fe_off + cell * 27 + t] = r;
  }
}

// grid (ceil(n_dof / 128), nbc)
__global__ void __launch_bounds__(128) k3v_apply_gather(DevGrid3 g, const double* __restrict__ FE, long long fe_stride,
                                                        long long fe_off, double* __restrict__ out, long long f_stride,
                                                        long long f_off, int b0) {
  const int i = blockIdx.x * 128 + threadIdx.x, b = blockIdx.y;
  if (i >= g.n_dof) return;
  const double* fe = FE + (long long)b * fe_stride + fe_off;
  double v = 0.0;
  for (int p = g.ap_ptr[i]; p < g.ap_ptr[i + 1]; ++p) v = fma(g.ap_w[p], fe[g.ap_code[p]], v);
  out[(long long)(b0 + b) * f_stride + f_off + i] = v;
}

}  // namespace landau3v
