// k3_ring.cuh -- K3: element matrices of the shifted weak form and their assembly into the batched CSR
// (SURVEY 8a rows a3 + a4; eq. 2.4, 73, 75, 87-89).
//
//   A_e[a][c] = sum_q w_q [ phi_a phi_c / dt + grad phi_a . D grad phi_c - (grad phi_a . K) phi_c ]       (= M/dt - J)
//
// One CTA owns one (batch entry, species) block (or a segment of its cells) and walks the grid's cells in panels of
// K3_PC; the element matrices of the last `rc` cells live in a shared-memory ring, and after every panel the CSR
// slots whose last contributing cell lies in that panel are gathered from the ring and written ONCE, in ascending
// slot order (coalesced streaming stores, no atomics, deterministic).  The schedule (em_*, as_*) is built on the
// host (host_setup.cpp, "K3 ring schedule").
//
// Element matrix = sum-factorised FP64 contraction on the DMMA pipe, one warp per cell.  With the tensor-product
// basis phi_a = l_a1(xi) l_a2(eta) and the 1-D product tables Pxy[ac][q] = l^(x)_a(q) l^(y)_c(q):
//
//   stage 1 (contract q2):  Y[a2c2][(rtab, q1)] = sum_{ztab, q2} Pz_ztab[a2c2][q2] * W_{ztab,rtab}[q2][q1]
//   stage 2 (contract q1):  A[a1c1][a2c2]       = sum_{rtab, q1} Pr_rtab[a1c1][q1] * Y[a2c2][(rtab, q1)]
//
//   rtab \ ztab |  P00z      P11z     P10z     P01z            W = w_q x { 1/dt, Drr sr^2, Dzz sz^2, Drz sr sz,
//   P00r        |  Wm        Wzz     -Wkz       .                          Kr sr, Kz sz }   (sr = 2/hr, sz = 2/hz)
//   P11r        |  Wrr        .        .        .
//   P10r        | -Wkr        .        .       Wrz
//   P01r        |   .         .       Wrz       .
//
// Both stages are m8n8k4 DMMAs whose A operands are CONSTANT fragments (16 registers per lane, loaded once); the
// stage-1 C fragments are exactly the stage-2 B fragments (the contraction index is only permuted, and the constant
// stage-2 A fragments are built with the same permutation), so the chain never leaves registers: 12 + 16 DMMAs per
// cell instead of ~14k scalar FMAs.  Works for Q2 and Q3 (tables zero-padded to 16 x 4).
#pragma once
#include "host_setup.hpp"

namespace landau {

struct K3Grid {  // device copy of one grid's K3 schedule
  int n_cells, nq, n1, rc, nsteps;
  const double *cell_sr, *cell_sz, *ip_w;
  const int *em_ptr, *em_n;
  const unsigned short* em_off;
  const int *as_ptr, *as_roff;
  const double* as_w;
};

struct K3Species {
  int grid;
  long long dk_off, v_off, n_ip;
};

constexpr int K3_THREADS = 256;

__global__ void __launch_bounds__(K3_THREADS, 3)
k3_ring(const K3Grid* __restrict__ grids, const K3Species* __restrict__ spec, int n_spec, int nseg,
        const double* __restrict__ frag, const double* __restrict__ DK, long long dk_stride, double inv_dt,
        double* __restrict__ vals, long long v_stride) {
  extern __shared__ __align__(16) double ring[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int gq = lane >> 2, tq = lane & 3;
  int bid = blockIdx.x;
  const int seg = bid % nseg;
  bid /= nseg;
  const int sidx = bid % n_spec, b = bid / n_spec;
  const K3Species sp = spec[sidx];
  const K3Grid g = grids[sp.grid];
  const int s_lo = (int)((long long)seg * g.nsteps / nseg), s_hi = (int)((long long)(seg + 1) * g.nsteps / nseg);
  if (s_lo >= s_hi) return;
  const int s_begin = max(0, s_lo - (g.rc / K3_PC - 1));

  double az[8], ar[8];
#pragma unroll
  for (int x = 0; x < 8; ++x) {
    az[x] = frag[x * 32 + lane];
    ar[x] = frag[(8 + x) * 32 + lane];
  }
  const int q1 = gq & 3, q2 = tq;
  const bool hi = gq >= 4;
  const bool valid = q1 < g.n1 && q2 < g.n1;
  const int qidx = q1 + g.n1 * q2;
  const double* dk = DK + (long long)b * dk_stride + sp.dk_off;
  double* out = vals + (long long)b * v_stride + sp.v_off;

  for (int s = s_begin; s < s_hi; ++s) {
#pragma unroll 1
    for (int cc = warp; cc < K3_PC; cc += K3_THREADS / 32) {
      const int cell = s * K3_PC + cc;
      if (cell >= g.n_cells) break;
      double w = 0.0, Drr = 0.0, Drz = 0.0, Dzz = 0.0, Kr = 0.0, Kz = 0.0;
      if (valid) {
        const long long ip = (long long)cell * g.nq + qidx;
        w = g.ip_w[ip];
        Drr = dk[ip];
        Drz = dk[sp.n_ip + ip];
        Dzz = dk[2 * sp.n_ip + ip];
        Kr = dk[3 * sp.n_ip + ip];
        Kz = dk[4 * sp.n_ip + ip];
      }
      const double sr = g.cell_sr[cell], sz = g.cell_sz[cell];
      const double wr = w * sr, wz = w * sz;
      const double Wm = w * inv_dt, Wrr = wr * sr * Drr, Wzz = wz * sz * Dzz, Wrz = wr * sz * Drz, Wkr = wr * Kr,
                   Wkz = wz * Kz;
      // stage-1 B fragments: B[k = q2][n = (rtab, q1)], rtab = 2 nt + (gq >= 4)
      const double b00 = hi ? Wrr : Wm, b01 = hi ? 0.0 : Wzz, b02 = hi ? 0.0 : -Wkz;
      const double b10 = hi ? 0.0 : -Wkr, b12 = hi ? Wrz : 0.0, b13 = hi ? 0.0 : Wrz;
      double y[2][2][2];
#pragma unroll
      for (int mt = 0; mt < 2; ++mt) {
        y[mt][0][0] = y[mt][0][1] = y[mt][1][0] = y[mt][1][1] = 0.0;
        dmma884(y[mt][0][0], y[mt][0][1], az[0 * 2 + mt], b00);
        dmma884(y[mt][1][0], y[mt][1][1], az[0 * 2 + mt], b10);
        dmma884(y[mt][0][0], y[mt][0][1], az[1 * 2 + mt], b01);
        dmma884(y[mt][1][0], y[mt][1][1], az[2 * 2 + mt], b12);
        dmma884(y[mt][0][0], y[mt][0][1], az[2 * 2 + mt], b02);
        dmma884(y[mt][1][0], y[mt][1][1], az[3 * 2 + mt], b13);
      }
      // stage 2: A[m = a1c1][n = a2c2]; k-step (nt, h) takes y[.][nt][h] as its B fragment
      double o[2][2][2];
#pragma unroll
      for (int mt2 = 0; mt2 < 2; ++mt2)
#pragma unroll
        for (int nt2 = 0; nt2 < 2; ++nt2) o[mt2][nt2][0] = o[mt2][nt2][1] = 0.0;
#pragma unroll
      for (int ks = 0; ks < 4; ++ks)
#pragma unroll
        for (int mt2 = 0; mt2 < 2; ++mt2)
#pragma unroll
          for (int nt2 = 0; nt2 < 2; ++nt2)
            dmma884(o[mt2][nt2][0], o[mt2][nt2][1], ar[ks * 2 + mt2], y[nt2][ks >> 1][ks & 1]);
      double* dst = ring + (cell % g.rc) * K3_RS;
#pragma unroll
      for (int mt2 = 0; mt2 < 2; ++mt2)
#pragma unroll
        for (int nt2 = 0; nt2 < 2; ++nt2)
#pragma unroll
          for (int h = 0; h < 2; ++h) dst[(2 * tq + h + 8 * nt2) * K3_LD + gq + 8 * mt2] = o[mt2][nt2][h];
    }
    __syncthreads();
    if (s >= s_lo) {
      const int e1 = g.em_ptr[s + 1];
      for (int e = g.em_ptr[s] + tid; e < e1; e += K3_THREADS) {
        const int n = g.em_n[e];
        const unsigned off = g.em_off[e];
        double v;
        if (off != 0xFFFFu) {
          v = ring[off];
        } else {
          v = 0.0;
          for (int p = g.as_ptr[n]; p < g.as_ptr[n + 1]; ++p) v = fma(g.as_w[p], ring[g.as_roff[p]], v);
        }
        __stcs(out + n, v);
      }
    }
    __syncthreads();
  }
}

}  // namespace landau
