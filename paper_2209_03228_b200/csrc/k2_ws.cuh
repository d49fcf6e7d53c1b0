// k2_ws.cuh -- K2 for many source columns, warp-specialised:
//
//   G_k[i, col] = sum_j U_k(i,j) * F_l[j, col]      seven (k,l) products, DMMA m8n8k4 (SASS: DMMA)
//
// Same CTA tile and shared-memory images as k2_gemm.cuh (TI field points x TC columns, source tiles of 16 points,
// B stages moved by one bulk async copy each, tensor tile stored in DMMA A-fragment order), but the two kinds of FP64
// work run in different warps and overlap:
//   * 8 consumer warps (two warpgroups, setmaxnreg 224) only wait on mbarriers, read fragments and issue DMMAs: the
//     160 accumulator registers per thread live with no tensor-evaluation state beside them (no spills);
//   * 4 producer warps (one warpgroup, setmaxnreg 64) evaluate the Landau tensor of the NEXT source tiles into a ring
//     of NA tensor buffers -- their long dependent DFMA chains fill the issue slots the DMMA stream leaves free -- and
//     one producer thread issues the bulk copies of the F stages.
// full/empty mbarrier pairs per B stage and per tensor buffer; no __syncthreads in the main loop.
// Producer lane (g = lane/4, t = lane%4) of producer warp w evaluates the pairs (i = 8u + g, j = 4w + t), u < TI/8:
// one source point per thread per tile, and every warp store of a tensor component is 32 consecutive doubles of the
// fragment image (bank-conflict free).
#pragma once
#include <cstdint>

namespace landau {

__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// register split after setmaxnreg.  Registers move inside the CTA's own pool (what the launch allocated: 384 threads
// x 168), so 256 consumer threads x CONS + 128 producer threads x PROD must not exceed 384 x 168 = 64512 -- a
// larger request makes setmaxnreg.inc wait forever.
#ifndef K2W_CONS_REGS
#define K2W_CONS_REGS 216
#define K2W_PROD_REGS 72
#endif
static_assert(256 * K2W_CONS_REGS + 128 * K2W_PROD_REGS <= 384 * 168, "setmaxnreg split exceeds the CTA register pool");
static_assert(K2W_CONS_REGS % 8 == 0 && K2W_PROD_REGS % 8 == 0, "setmaxnreg takes multiples of 8");

template <int WI_T, int WC_T, int WGI, int WGC, int NST, int NA>
struct K2W {
  static constexpr int NCONS = WGI * WGC;        // consumer warps (must be 8: two warpgroups)
  static constexpr int NPROD = 4;                // producer warps (one warpgroup)
  static constexpr int NTHREADS = 32 * (NCONS + NPROD);
  static constexpr int TI = 8 * WI_T * WGI;
  static constexpr int TC = 8 * WC_T * WGC;
  static constexpr int STAGE_DOUBLES = 3 * TC * K2G_TJ;
  static constexpr int A_CS = (TI / 8) * 4 * 32;  // doubles per tensor component in one buffer
  static constexpr int A_DOUBLES = 5 * A_CS;
  static constexpr int NU = TI / 8;               // pairs per producer thread per source tile
  static constexpr size_t SMEM_BYTES = (size_t)(NST * STAGE_DOUBLES + NA * A_DOUBLES) * 8 + (2 * NST + 2 * NA) * 8;
  static_assert(NCONS == 8, "two consumer warpgroups");
};

template <int WI_T, int WC_T, int WGI, int WGC, int NST, int NA>
__global__ void __launch_bounds__(K2W<WI_T, WC_T, WGI, WGC, NST, NA>::NTHREADS, 1)
k2_inner_ws(const double* __restrict__ ip_r, const double* __restrict__ ip_z, int n_i, int j0, int njt,
            const double* __restrict__ F, int ncols, double* __restrict__ G, long long g_split_stride, int gcol0) {
  using C = K2W<WI_T, WC_T, WGI, WGC, NST, NA>;
  extern __shared__ __align__(128) double smem_w[];
  double* sB = smem_w;                                // [NST][3][TC][16]
  double* sA = smem_w + NST * C::STAGE_DOUBLES;       // [NA][5][TI/8][4][32]
  uint64_t* fullB = reinterpret_cast<uint64_t*>(sA + NA * C::A_DOUBLES);
  uint64_t* emptyB = fullB + NST;
  uint64_t* fullA = emptyB + NST;
  uint64_t* emptyA = fullA + NA;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int i0 = blockIdx.x * C::TI;
  const int per = (njt + gridDim.z - 1) / gridDim.z;
  const int t0 = blockIdx.z * per, t1 = min(t0 + per, njt);
  const int nt = max(t1 - t0, 0);
  const double* Fct = F + (long long)blockIdx.y * njt * C::STAGE_DOUBLES;

  if (tid == 0) {
    for (int s = 0; s < NST; ++s) {
      mbar_init(&fullB[s], 1);
      mbar_init(&emptyB[s], C::NCONS);
    }
    for (int s = 0; s < NA; ++s) {
      mbar_init(&fullA[s], C::NPROD * 32);
      mbar_init(&emptyA[s], C::NCONS);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();

  if (warp >= C::NCONS) {
    // =========================================== producers ===========================================
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(K2W_PROD_REGS));
    const int pw = warp - C::NCONS, gq = lane >> 2, tq = lane & 3;
    const int jl = pw * 4 + tq;
    double ri[C::NU], zi[C::NU];
#pragma unroll
    for (int u = 0; u < C::NU; ++u) {
      const int ig = min(i0 + u * 8 + gq, n_i - 1);
      ri[u] = ip_r[ig];
      zi[u] = ip_z[ig];
    }
    double rj = 0.0, zj = 0.0;
    if (nt > 0) {
      rj = ip_r[j0 + t0 * K2G_TJ + jl];
      zj = ip_z[j0 + t0 * K2G_TJ + jl];
    }
    for (int tt = 0; tt < nt; ++tt) {
      if (tid == C::NCONS * 32) {  // F stage of this step
        const int stage = tt % NST;
        if (tt >= NST) mbar_wait(&emptyB[stage], ((tt / NST) - 1) & 1);
        mbar_expect_tx(&fullB[stage], C::STAGE_DOUBLES * 8);
        bulk_g2s(sB + stage * C::STAGE_DOUBLES, Fct + (long long)(t0 + tt) * C::STAGE_DOUBLES, C::STAGE_DOUBLES * 8,
                 &fullB[stage]);
      }
      const double rjc = rj, zjc = zj;
      if (tt + 1 < nt) {  // next tile's source point, in flight during this tile's evaluation
        rj = ip_r[j0 + (t0 + tt + 1) * K2G_TJ + jl];
        zj = ip_z[j0 + (t0 + tt + 1) * K2G_TJ + jl];
      }
      const int buf = tt % NA;
      if (tt >= NA) mbar_wait(&emptyA[buf], ((tt / NA) - 1) & 1);
      double* dst = sA + buf * C::A_DOUBLES + ((pw << 5) | lane);
#pragma unroll
      for (int u = 0; u < C::NU; ++u) {
        const Tensor5 U = landau_tensor_2v(ri[u], zi[u], rjc, zjc);
        double* d = dst + (u << 7);  // block (i block u, k4 = pw): ((u*4 + pw) << 5) + lane
        d[0] = U.UDrr;
        d[C::A_CS] = U.UDrz;
        d[2 * C::A_CS] = U.UDzz;
        d[3 * C::A_CS] = U.UKrr;
        d[4 * C::A_CS] = U.UKzr;
      }
      mbar_arrive(&fullA[buf]);
    }
  } else {
    // =========================================== consumers ===========================================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(K2W_CONS_REGS));
    const int wi = warp / WGC, wc = warp - wi * WGC;
    const int gq = lane >> 2, tq = lane & 3;
    double acc[WI_T][WC_T][5][2];
#pragma unroll
    for (int x = 0; x < WI_T; ++x)
#pragma unroll
      for (int n = 0; n < WC_T; ++n)
#pragma unroll
        for (int k = 0; k < 5; ++k) acc[x][n][k][0] = acc[x][n][k][1] = 0.0;

    for (int tt = 0; tt < nt; ++tt) {
      const int stage = tt % NST, buf = tt % NA;
      mbar_wait(&fullA[buf], (tt / NA) & 1);
      mbar_wait(&fullB[stage], (tt / NST) & 1);
      const double* A = sA + buf * C::A_DOUBLES + lane;
      const double* Bst = sB + stage * C::STAGE_DOUBLES;
#pragma unroll
      for (int ks = 0; ks < 4; ++ks) {
        double a[WI_T][5];
#pragma unroll
        for (int x = 0; x < WI_T; ++x)
#pragma unroll
          for (int k = 0; k < 5; ++k) a[x][k] = A[k * C::A_CS + (((wi * WI_T + x) * 4 + ks) << 5)];
#pragma unroll
        for (int n = 0; n < WC_T; ++n) {
          const int cl = (wc * WC_T + n) * 8 + gq;
          const double* bp = Bst + cl * 16 + (((ks ^ (gq & 3)) << 2) | tq);
          const double wf = bp[0], wfr = bp[C::TC * 16], wfz = bp[2 * C::TC * 16];
#pragma unroll
          for (int x = 0; x < WI_T; ++x) {
            dmma884(acc[x][n][0][0], acc[x][n][0][1], a[x][0], wf);
            dmma884(acc[x][n][1][0], acc[x][n][1][1], a[x][1], wf);
            dmma884(acc[x][n][2][0], acc[x][n][2][1], a[x][2], wf);
            dmma884(acc[x][n][3][0], acc[x][n][3][1], a[x][3], wfr);
            dmma884(acc[x][n][4][0], acc[x][n][4][1], a[x][4], wfr);
            dmma884(acc[x][n][3][0], acc[x][n][3][1], a[x][1], wfz);
            dmma884(acc[x][n][4][0], acc[x][n][4][1], a[x][2], wfz);
          }
        }
      }
      __syncwarp();
      if (lane == 0) {
        mbar_arrive(&emptyA[buf]);
        mbar_arrive(&emptyB[stage]);
      }
    }
    // C fragment: row gq (field point), columns 2 tq, 2 tq + 1
#pragma unroll
    for (int x = 0; x < WI_T; ++x) {
      const int i = i0 + (wi * WI_T + x) * 8 + gq;
      if (i < n_i) {
#pragma unroll
        for (int n = 0; n < WC_T; ++n)
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            const int col = blockIdx.y * C::TC + (wc * WC_T + n) * 8 + 2 * tq + h;
            if (col < ncols) {
              double* dst = G + blockIdx.z * g_split_stride + ((long long)(gcol0 + col) * 5) * n_i + i;
#pragma unroll
              for (int k = 0; k < 5; ++k) dst[(long long)k * n_i] = acc[x][n][k][h];
            }
          }
      }
    }
  }
}

}  // namespace landau
