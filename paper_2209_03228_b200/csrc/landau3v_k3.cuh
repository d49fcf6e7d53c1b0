// landau3v_k3.cuh -- K3 of the 3V variant: element matrices on the FP64 MMA pipe, then the CSR gather.
//
// With alpha_a(q) = w_q (phi_a / dt - grad phi_a . K) and beta_a(q) = w_q D grad phi_a (a 3-vector) the element matrix of
// M/dt - J is ONE dense contraction per cell,
//
//     A[a][c] = sum_q ( alpha_a(q) phi_c(q) + beta_a(q) . grad phi_c(q) ) = sum_{(q, k)} L[a][(q, k)] R[(q, k)][c],   k = 0..3,
//
// a 27 x 108 x 27 product whose right factor R (basis values and reference gradients at the 27 Gauss points) is CONSTANT.
// It is issued as mma.sync.m8n8k4.f64 with one warp per cell: k-step q contracts the four components k of point q, lane
// (g, t) forms L[8 mt + g][(q, t)] from four table values and four per-cell coefficients (a 4-term dot product: t = 0 gives
// alpha, t = 1..3 the components of beta), the R fragments come from a shared-memory table: 432 DMMAs per cell (110 k
// FMA slots) against 256 k scalar FMAs for the 13 weight fields taken one by one, and against the first version of this
// step (k3v_assemble, every CSR slot integrating its own entries: 43.7 ms on the paper's 3V problem at batch 32).
// The matrices go to a scratch array [entry][species][cell][27 x 27]; k3v_gather sums the entries of every CSR slot with the
// constraint weights and writes each value once (no atomics, deterministic).
#pragma once
#include "landau3v_dmma.cuh"

namespace landau3v {

// one launch covers every species: blockIdx.z picks the species, its grid comes from a device table
struct Spec3 {
  int grid;
  long long dk_off, em_off, v_off;
};

constexpr int K3E_WARPS = 4;
// dynamic shared memory of k3v_elem_matrix: tab4 [27][32][4] | coef [warps][27][4][4]
constexpr size_t K3E_SMEM = (27 * 32 * 4 + K3E_WARPS * 27 * 16) * sizeof(double);

// Persistent grid: every warp strides through the (species, entry, cell) items; the basis table is loaded once per CTA.
// (The first version started one CTA per four cells and reloaded 55 KB of tables each time.)
__global__ void __launch_bounds__(K3E_WARPS * 32) k3v_elem_matrix(const DevGrid3* __restrict__ grids, const Spec3* __restrict__ spec,
                                                                 int n_spec, int nbc, int max_cells,
                                                                 const Tables3* __restrict__ tab, const double* __restrict__ DK,
                                                                 long long dk_stride, double inv_dt, double* __restrict__ EM,
                                                                 long long em_stride) {
  extern __shared__ __align__(16) double sm3[];
  double* tab4 = sm3;                  // [q][a (32, zero padded)][B, dBx, dBy, dBz]; also the R fragments: R[(q, t)][8 nt + g]
                                       // = tab4[q][8 nt + g][t] = tab4[q * 128 + nt * 32 + lane]
  double* coef = tab4 + 27 * 32 * 4;   // [warp][q][t][4]
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, gq = lane >> 2, t = lane & 3;
  for (int e = tid; e < 27 * 32; e += K3E_WARPS * 32) {
    const int q = e / 32, a = e % 32;
    const bool ok = a < 27;
    tab4[e * 4] = ok ? tab->B[q * 27 + a] : 0.0;
    tab4[e * 4 + 1] = ok ? tab->dBx[q * 27 + a] : 0.0;
    tab4[e * 4 + 2] = ok ? tab->dBy[q * 27 + a] : 0.0;
    tab4[e * 4 + 3] = ok ? tab->dBz[q * 27 + a] : 0.0;
  }
  __syncthreads();
  double* cw = coef + warp * 27 * 16;
  const long long n_items = (long long)n_spec * nbc * max_cells;
  for (long long item = (long long)blockIdx.x * K3E_WARPS + warp; item < n_items; item += (long long)gridDim.x * K3E_WARPS) {
    const int cell = (int)(item % max_cells), b = (int)((item / max_cells) % nbc), sidx = (int)(item / ((long long)max_cells * nbc));
    const Spec3 sp = spec[sidx];
    const DevGrid3& g = grids[sp.grid];
    if (cell >= g.n_cells) continue;
    __syncwarp();
    // per-cell coefficients: lane q < 27 loads the point's weight, D and K
    if (lane < 27) {
      const long long N = g.n_ip;
      const int ip = cell * 27 + lane;
      const double* dk = DK + (long long)b * dk_stride + sp.dk_off + ip;
      const double sc = 2.0 / g.cell_h[cell], w = g.ip_w[ip], ws = w * sc, wss = ws * sc;
      const double dxx = wss * dk[0], dxy = wss * dk[N], dxz = wss * dk[2 * N], dyy = wss * dk[3 * N], dyz = wss * dk[4 * N],
                   dzz = wss * dk[5 * N];
      double* c = cw + lane * 16;
      c[0] = w * inv_dt;
      c[1] = -ws * dk[6 * N];
      c[2] = -ws * dk[7 * N];
      c[3] = -ws * dk[8 * N];
      c[4] = 0.0;
      c[5] = dxx;
      c[6] = dxy;
      c[7] = dxz;
      c[8] = 0.0;
      c[9] = dxy;
      c[10] = dyy;
      c[11] = dyz;
      c[12] = 0.0;
      c[13] = dxz;
      c[14] = dyz;
      c[15] = dzz;
    }
    __syncwarp();
    double acc[4][4][2];
#pragma unroll
    for (int mt = 0; mt < 4; ++mt)
#pragma unroll
      for (int nt = 0; nt < 4; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = 0.0;
#pragma unroll 1
    for (int q = 0; q < 27; ++q) {
      const double2 c01 = *reinterpret_cast<const double2*>(cw + q * 16 + t * 4), c23 = *reinterpret_cast<const double2*>(cw + q * 16 + t * 4 + 2);
      double l[4];
#pragma unroll
      for (int mt = 0; mt < 4; ++mt) {
        const double* tp = tab4 + (q * 32 + 8 * mt + gq) * 4;
        const double2 t01 = *reinterpret_cast<const double2*>(tp), t23 = *reinterpret_cast<const double2*>(tp + 2);
        l[mt] = fma(c01.x, t01.x, fma(c01.y, t01.y, fma(c23.x, t23.x, c23.y * t23.y)));
      }
#pragma unroll
      for (int nt = 0; nt < 4; ++nt) {
        const double r = tab4[q * 128 + nt * 32 + lane];
#pragma unroll
        for (int mt = 0; mt < 4; ++mt) dmma3(acc[mt][nt][0], acc[mt][nt][1], l[mt], r);
      }
    }
    // C fragment: lane (g, t) holds A[8 mt + g][8 nt + 2 t + h]
    double* dst = EM + (long long)b * em_stride + sp.em_off + (long long)cell * 729;
#pragma unroll
    for (int mt = 0; mt < 4; ++mt) {
      const int a = 8 * mt + gq;
      if (a < 27) {
#pragma unroll
        for (int nt = 0; nt < 4; ++nt)
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            const int c = 8 * nt + 2 * t + h;
            if (c < 27) dst[a * 27 + c] = acc[mt][nt][h];
          }
      }
    }
  }
}

// grid (ceil(max nnz / 256), ceil(nbc / K3G_BT), S): one thread per CSR slot and K3G_BT batch entries -- the slot's list of
// (weight, matrix entry) is read once for all of them and their loads are independent
constexpr int K3G_BT = 8;
__global__ void __launch_bounds__(256) k3v_gather(const DevGrid3* __restrict__ grids, const Spec3* __restrict__ spec, int nbc,
                                                  const double* __restrict__ EM, long long em_stride, double* __restrict__ vals,
                                                  long long v_stride) {
  const Spec3 sp = spec[blockIdx.z];
  const DevGrid3& g = grids[sp.grid];
  const int n = blockIdx.x * 256 + threadIdx.x, b0 = blockIdx.y * K3G_BT;
  if (n >= g.nnz) return;
  const double* em = EM + (long long)b0 * em_stride + sp.em_off;
  double v[K3G_BT];
#pragma unroll
  for (int k = 0; k < K3G_BT; ++k) v[k] = 0.0;
  const int p1 = g.as_ptr[n + 1];
  if (b0 + K3G_BT <= nbc) {
    for (int p = g.as_ptr[n]; p < p1; ++p) {
      const double w = g.as_w[p];
      const double* src = em + g.as_code[p];
#pragma unroll
      for (int k = 0; k < K3G_BT; ++k) v[k] = fma(w, src[k * em_stride], v[k]);
    }
  } else {
    for (int p = g.as_ptr[n]; p < p1; ++p) {
      const double w = g.as_w[p];
      const double* src = em + g.as_code[p];
#pragma unroll
      for (int k = 0; k < K3G_BT; ++k)
        if (b0 + k < nbc) v[k] = fma(w, src[k * em_stride], v[k]);
    }
  }
  double* dst = vals + (long long)b0 * v_stride + sp.v_off + n;
#pragma unroll
  for (int k = 0; k < K3G_BT; ++k)
    if (b0 + k < nbc) __stcs(dst + k * v_stride, v[k]);
}

}  // namespace landau3v
