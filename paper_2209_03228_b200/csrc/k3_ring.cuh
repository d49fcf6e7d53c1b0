// k3_ring.cuh -- K3: element matrices of the shifted weak form and their assembly into the batched CSR
// (SURVEY 8a rows a3 + a4; eq. 2.4, 73, 75, 87-89).
//
//   A_e[a][c] = sum_q w_q [ phi_a phi_c / dt + grad phi_a . D grad phi_c - (grad phi_a . K) phi_c ]       (= M/dt - J)
//
// One CTA owns one (batch entry, species) block (or a segment of its cells) and walks the grid's cells in panels of
// K3_PC; the element matrices of the last `rc` cells live in a shared-memory ring, and after every panel the CSR
// slots whose last contributing cell lies in that panel are gathered from the ring and written ONCE, in ascending
// slot order (coalesced streaming stores, no atomics, deterministic).  The schedule (em_*, as_*) is built on the
// host (host_setup.cpp, "K3 ring schedule"): packed 4-byte words for the ~88 % of slots fed by one element-matrix
// entry, 16-byte records for shared-node slots (<= 4 unit-weight entries), index lists for hanging-node slots, each
// list homogeneous so that warps do not diverge.  The quadrature-point data (w, D, K) of the next panel is fetched
// while the current panel is being emitted.
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
// Both stages are m8n8k4 DMMAs whose A operands are CONSTANT fragments (16 doubles per lane, kept in shared memory); the
// stage-1 C fragments are exactly the stage-2 B fragments (the contraction index is only permuted, and the constant
// stage-2 A fragments are built with the same permutation), so the chain never leaves registers: 12 + 16 DMMAs per
// cell instead of ~14k scalar FMAs.  Works for Q2 and Q3 (tables zero-padded to 16 x 4).
#pragma once
#include "host_setup.hpp"

namespace landau {

struct K3Grid {  // device copy of one grid's K3 schedule (host_setup.hpp, "K3 ring schedule")
  int n_cells, nq, n1, rc, nsteps;
  const double *cell_sr, *cell_sz, *ip_w;
  const int *em_ptr, *em_base, *emg;
  const unsigned* em1;
  const uint4* em4;
  const int *as_ptr, *as_roff;
  const double* as_w;
  const int *cell_pos, *halo_begin;
};

struct K3Species {
  int grid;
  long long dk_off, v_off, n_ip;
};

constexpr int K3_THREADS = 256;
constexpr int K3_CPW = K3_PC / (K3_THREADS / 32);  // cells per warp per step
constexpr int K3_EB = 8;                            // emission: descriptor words per thread per batch

__device__ __forceinline__ double k3_lds(unsigned addr) {
  double v;
  asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
  return v;
}

// dynamic shared memory: ring [rc][K3_RS] | zero pad [8] | constant fragments [16][32]
__host__ __device__ constexpr size_t k3_smem_bytes(int rc) { return ((size_t)rc * K3_RS + 8 + 16 * 32) * sizeof(double); }

__global__ void __launch_bounds__(K3_THREADS, 4)
k3_ring(const K3Grid* __restrict__ grids, const K3Species* __restrict__ spec, int n_spec, int n_whole, int nseg,
        const double* __restrict__ frag, const double* __restrict__ DK, long long dk_stride, double inv_dt,
        double* __restrict__ vals, long long v_stride) {
  extern __shared__ __align__(16) double ring[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int gq = lane >> 2, tq = lane & 3;
  // blocks [0, n_whole): one (entry, species) block each; later blocks: the remaining (entry, species) blocks cut into
  // nseg segments of steps each (landau_api.cu, assemble_chunk: fills the last wave / small batches)
  int bid = blockIdx.x, seg = 0;
  if (bid >= n_whole) {
    const int j = bid - n_whole;
    seg = j % nseg;
    bid = n_whole + j / nseg;
  } else {
    nseg = 1;
  }
  const int sidx = bid % n_spec, b = bid / n_spec;
  const K3Species sp = spec[sidx];
  const K3Grid* __restrict__ g = grids + sp.grid;
  const int nsteps = g->nsteps, rc = g->rc, n_cells = g->n_cells, n1 = g->n1, nq = g->nq;
  const int s_lo = (int)((long long)seg * nsteps / nseg), s_hi = (int)((long long)(seg + 1) * nsteps / nseg);
  if (s_lo >= s_hi) return;
  const int s_begin = g->halo_begin[s_lo];

  const unsigned ring_s = smem_u32(ring);
  double* zero_pad = ring + rc * K3_RS;
  double* sfrag = zero_pad + 8;
  if (tid < 8) zero_pad[tid] = 0.0;
  for (int e = tid; e < 16 * 32; e += K3_THREADS) sfrag[e] = frag[e];
  const double* fr = sfrag + lane;

  const int q1 = gq & 3, q2 = tq;
  const bool hi = gq >= 4;
  const bool valid = q1 < n1 && q2 < n1;
  const int qidx = q1 + n1 * q2;
  const double* __restrict__ dk = DK + (long long)b * dk_stride + sp.dk_off;
  const double* __restrict__ ip_w = g->ip_w;
  const double* __restrict__ cell_sr = g->cell_sr;
  const double* __restrict__ cell_sz = g->cell_sz;
  double* __restrict__ out = vals + (long long)b * v_stride + sp.v_off;
  const int S1 = nsteps + 1;

  // this lane's quadrature-point data of the warp's cells, fetched one step ahead of its use
  double wv[K3_CPW][6], sc[K3_CPW][2];
  int pos[K3_CPW];
  const int* __restrict__ cell_pos = g->cell_pos;
  auto fetch = [&](int s) {
#pragma unroll
    for (int u = 0; u < K3_CPW; ++u) {
      const int cell = s * K3_PC + warp + u * (K3_THREADS / 32);
      const bool ok = cell < n_cells;
      const long long ip = (long long)(ok ? cell : 0) * nq + (valid ? qidx : 0);
      const double m = (ok && valid) ? 1.0 : 0.0;
      wv[u][0] = m * ip_w[ip];
#pragma unroll
      for (int k = 0; k < 5; ++k) wv[u][1 + k] = dk[k * sp.n_ip + ip];
      sc[u][0] = cell_sr[ok ? cell : 0];
      sc[u][1] = cell_sz[ok ? cell : 0];
      pos[u] = cell_pos[ok ? cell : 0];
    }
  };
  fetch(s_begin);
  // list bounds of the panel to emit, loaded one step ahead: em1 [pa[0], pa[1]), em4 [pa[2], pa[3]), slot base pa[4],
  // general list [pa[5], pa[6])
  int pa[7];
  auto fetch_bounds = [&](int s) {
    pa[0] = g->em_ptr[s];
    pa[1] = g->em_ptr[s + 1];
    pa[2] = g->em_ptr[S1 + s];
    pa[3] = g->em_ptr[S1 + s + 1];
    pa[4] = g->em_base[s];
    pa[5] = g->em_ptr[2 * S1 + s];
    pa[6] = g->em_ptr[2 * S1 + s + 1];
  };
  fetch_bounds(s_begin);
  __syncthreads();

  for (int s = s_begin; s < s_hi; ++s) {
#pragma unroll
    for (int u = 0; u < K3_CPW; ++u) {
      const int cell = s * K3_PC + warp + u * (K3_THREADS / 32);
      if (cell < n_cells) {
        const double w = wv[u][0], sr = sc[u][0], sz = sc[u][1];
        const double wr = w * sr, wz = w * sz;
        const double Wm = w * inv_dt, Wrr = wr * sr * wv[u][1], Wrz = wr * sz * wv[u][2], Wzz = wz * sz * wv[u][3],
                     Wkr = wr * wv[u][4], Wkz = wz * wv[u][5];
        // stage-1 B fragments: B[k = q2][n = (rtab, q1)], rtab = 2 nt + (gq >= 4)
        const double b00 = hi ? Wrr : Wm, b01 = hi ? 0.0 : Wzz, b02 = hi ? 0.0 : -Wkz;
        const double b10 = hi ? 0.0 : -Wkr, b12 = hi ? Wrz : 0.0, b13 = hi ? 0.0 : Wrz;
        double y[2][2][2];
#pragma unroll
        for (int mt = 0; mt < 2; ++mt) {
          y[mt][0][0] = y[mt][0][1] = y[mt][1][0] = y[mt][1][1] = 0.0;
          dmma884(y[mt][0][0], y[mt][0][1], fr[(0 * 2 + mt) * 32], b00);
          dmma884(y[mt][1][0], y[mt][1][1], fr[(0 * 2 + mt) * 32], b10);
          dmma884(y[mt][0][0], y[mt][0][1], fr[(1 * 2 + mt) * 32], b01);
          dmma884(y[mt][1][0], y[mt][1][1], fr[(2 * 2 + mt) * 32], b12);
          dmma884(y[mt][0][0], y[mt][0][1], fr[(2 * 2 + mt) * 32], b02);
          dmma884(y[mt][1][0], y[mt][1][1], fr[(3 * 2 + mt) * 32], b13);
        }
        // stage 2: A[m = a1c1][n = a2c2]; k-step ks = (nt, h) takes y[.][nt][h] as its B fragment
        double o[2][2][2];
#pragma unroll
        for (int mt2 = 0; mt2 < 2; ++mt2)
#pragma unroll
          for (int nt2 = 0; nt2 < 2; ++nt2) o[mt2][nt2][0] = o[mt2][nt2][1] = 0.0;
#pragma unroll
        for (int ks = 0; ks < 4; ++ks)
#pragma unroll
          for (int mt2 = 0; mt2 < 2; ++mt2) {
            const double a = fr[(8 + ks * 2 + mt2) * 32];
#pragma unroll
            for (int nt2 = 0; nt2 < 2; ++nt2) dmma884(o[mt2][nt2][0], o[mt2][nt2][1], a, y[nt2][ks >> 1][ks & 1]);
          }
        double* dst = ring + pos[u] * K3_RS;
#pragma unroll
        for (int mt2 = 0; mt2 < 2; ++mt2)
#pragma unroll
          for (int nt2 = 0; nt2 < 2; ++nt2)
#pragma unroll
            for (int h = 0; h < 2; ++h) dst[k3_entry_offset(2 * tq + h + 8 * nt2, gq + 8 * mt2)] = o[mt2][nt2][h];
      }
    }
    if (s + 1 < s_hi) fetch(s + 1);
    // first batch of this panel's emission descriptors: issued before the barrier, consumed after it
    const bool emit = s >= s_lo;
    const int base = pa[4];
    const unsigned* __restrict__ em1 = g->em1;
    const uint4* __restrict__ em4 = g->em4;
    const int e1_lo = pa[0] + tid, e1_hi = emit ? pa[1] : 0;
    const int e4_lo = pa[2] + tid, e4_hi = emit ? pa[3] : 0;
    const int eg_lo = pa[5] + tid, eg_hi = pa[6];
    unsigned wd[K3_EB];
    uint4 d4[2];
#pragma unroll
    for (int k = 0; k < K3_EB; ++k) {
      const int e = e1_lo + k * K3_THREADS;
      wd[k] = e < e1_hi ? __ldg(em1 + e) : 0xFFFFFFFFu;
    }
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      const int e = e4_lo + k * K3_THREADS;
      d4[k] = e < e4_hi ? __ldg(em4 + e) : make_uint4(0xFFFFFFFFu, 0, 0, 0);
    }
    if (s + 1 < s_hi) fetch_bounds(s + 1);
    __syncthreads();
    if (emit) {
      double* __restrict__ outb = out + base;
      // one contribution, weight 1
      for (int e0 = e1_lo;;) {
#pragma unroll
        for (int k = 0; k < K3_EB; ++k)
          if (wd[k] != 0xFFFFFFFFu)  // 32-bit shared address, one widening multiply-add for the global one
            __stcs(outb + (wd[k] & ((1u << K3_NBITS) - 1)), k3_lds(ring_s + ((wd[k] >> (K3_NBITS - 3)) & ~7u)));
        e0 += K3_THREADS * K3_EB;
        if (e0 >= e1_hi) break;
#pragma unroll
        for (int k = 0; k < K3_EB; ++k) {
          const int e = e0 + k * K3_THREADS;
          wd[k] = e < e1_hi ? __ldg(em1 + e) : 0xFFFFFFFFu;
        }
      }
      // 2..4 contributions, weight 1
      for (int e0 = e4_lo;;) {
#pragma unroll
        for (int k = 0; k < 2; ++k)
          if (d4[k].x != 0xFFFFFFFFu) {
            const double v = ((k3_lds(ring_s + (d4[k].y & 0xFFFFu) * 8) + k3_lds(ring_s + (d4[k].y >> 16) * 8)) +
                              k3_lds(ring_s + (d4[k].z & 0xFFFFu) * 8)) +
                             k3_lds(ring_s + (d4[k].z >> 16) * 8);
            __stcs(outb + d4[k].x, v);
          }
        e0 += K3_THREADS * 2;
        if (e0 >= e4_hi) break;
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          const int e = e0 + k * K3_THREADS;
          d4[k] = e < e4_hi ? __ldg(em4 + e) : make_uint4(0xFFFFFFFFu, 0, 0, 0);
        }
      }
      {  // general: hanging-node weights
        const int* __restrict__ emg = g->emg;
        const int* __restrict__ as_ptr = g->as_ptr;
        const int* __restrict__ as_roff = g->as_roff;
        const double* __restrict__ as_w = g->as_w;
        for (int e = eg_lo; e < eg_hi; e += K3_THREADS) {
          const int n = emg[e];
          double v = 0.0;
          for (int p = as_ptr[n]; p < as_ptr[n + 1]; ++p) v = fma(as_w[p], ring[as_roff[p]], v);
          __stcs(out + n, v);
        }
      }
    }
    __syncthreads();
  }
}

}  // namespace landau
