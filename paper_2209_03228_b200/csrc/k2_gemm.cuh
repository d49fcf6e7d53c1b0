// k2_gemm.cuh -- K2 for many source columns: the inner integral as an FP64
// contraction whose A operand (the Landau tensor) is generated ONCE per CTA per (i,j) tile and shared by all warps.
//
//   G_k[i, col] = sum_j U_k(i,j) * F_l[j, col]      seven (k,l) products, DMMA m8n8k4 (SASS: DMMA)
//
// CTA tile: TI field points x TC columns, K loop over source tiles of 16 points.
//   * B operand (source fields F): global layout is already the shared-memory image of a stage
//     ([col tile][j tile][comp 3][col in tile][16 j, 4-blocks XOR-swizzled by col&3]), so one elected thread moves a
//     stage with ONE bulk async copy (TMA, cp.async.bulk -> SASS UBLKCP) that signals an mbarrier; NST stages.
//   * A operand (tensor): all threads evaluate the TI x 16 tensor tile of the NEXT step while the DMMAs of the
//     current step are in flight (other warps), and store it in DMMA A-fragment order ([comp][i block][k4][lane]),
//     double buffered; every warp then reads its fragments with conflict-free contiguous 256-byte loads.
//   * one __syncthreads per 16 source points.
// Warp tile: (8 WI_T) field points x (8 WC_T) columns; WGI x WGC warps.
#pragma once
#include <cstdint>

namespace landau {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile(
        "{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
  } while (!ok);
}

template <int WI_T, int WC_T, int WGI, int WGC, int NST>
struct K2G {
  static constexpr int P_WI_T = WI_T, P_WC_T = WC_T, P_WGI = WGI, P_WGC = WGC, P_NST = NST;
  static constexpr int NTHREADS = 32 * WGI * WGC;
  static constexpr int TI = 8 * WI_T * WGI;
  static constexpr int TC = 8 * WC_T * WGC;
  static constexpr int STAGE_DOUBLES = 3 * TC * K2G_TJ;
  static constexpr int A_DOUBLES = 5 * (TI / 8) * 4 * 32;  // one buffer
  static constexpr int PAIRS_PER_THREAD = TI * K2G_TJ / NTHREADS;
  static constexpr int ACC_PER_THREAD = WI_T * WC_T * 10;
  static constexpr int TAB_DOUBLES = 4 * LANDAU_ELLIP_TAB_BINADES * (LANDAU_ELLIP_TAB_DEG + 1) * 4;
  static constexpr int XY_DOUBLES = 4 * 2 * K2G_TJ;  // ring of four source-tile coordinate blocks (r[16], z[16])
  static constexpr size_t SMEM_BYTES =
      (size_t)(NST * STAGE_DOUBLES + 2 * A_DOUBLES + TAB_DOUBLES + XY_DOUBLES) * 8 + NST * 8;
  static_assert(TI * K2G_TJ % NTHREADS == 0, "tensor tile must divide over the threads");
  static_assert((NTHREADS / 32) % 4 == 0, "warps must cover whole groups of the four k4 blocks");
};

template <int WI_T, int WC_T, int WGI, int WGC, int NST>
__global__ void __launch_bounds__(32 * WGI * WGC, 1)
k2_inner_gemm(const double* __restrict__ ip_r, const double* __restrict__ ip_z, int n_i, int j0, int njt,
              const double* __restrict__ F, int ncols, double* __restrict__ G, long long g_split_stride, int gcol0,
              int stream_itiles, int stream_tiles, double* __restrict__ part_buf, int part_stride,
              int* __restrict__ part_count) {
  using C = K2G<WI_T, WC_T, WGI, WGC, NST>;
  extern __shared__ __align__(128) double smem_g[];
  double* smem = smem_g;
  double* sB = smem;                                  // [NST][3][TC][16]
  double* sA = smem + NST * C::STAGE_DOUBLES;         // [2][5][TI/8][4][32]
  double* sTab = sA + 2 * C::A_DOUBLES;               // elliptic table T (13 KB), copied once
  double* sXY = sTab + C::TAB_DOUBLES;                // [4][2][16] source-point coordinates, filled by cp.async
  uint64_t* full = reinterpret_cast<uint64_t*>(sXY + C::XY_DOUBLES);

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wi = warp / WGC, wc = warp - wi * WGC;
  const int gq = lane >> 2, tq = lane & 3;
  // Work of this CTA.  Grid mode (stream_tiles == 0): one segment = tile (blockIdx.x, blockIdx.y), source tiles of
  // j-split blockIdx.z, plain stores into split plane blockIdx.z.
  // Stream mode: P = gridDim.x persistent CTAs, tiles ordered column tile slowest.  CTA p first takes the whole tiles
  // p, p + P, .. of the q = T / P full waves (resident CTAs walk the same F column tile in step: L2 reuse as in grid
  // mode); the r = T mod P tiles of the last, partial wave are cut evenly: their r * njt source-tile steps are shared
  // by all P CTAs.  A CTA that holds only part of a tile dumps its accumulators to `part_buf`; the CTA that arrives
  // last at the tile's counter adds the parts IN PART ORDER and stores the tile (deterministic, no atomics on G).
  long long w0, w1;
  int seg_k = 0, seg_q = 0;
  if (stream_tiles) {
    seg_q = stream_tiles / (int)gridDim.x;
    const long long R = (long long)(stream_tiles - seg_q * (int)gridDim.x) * njt;
    w0 = R * blockIdx.x / gridDim.x;
    w1 = R * (blockIdx.x + 1) / gridDim.x;
  } else {
    const int per = (njt + gridDim.z - 1) / gridDim.z;
    const int ta = blockIdx.z * per, tb = min(ta + per, njt);
    w0 = ta;
    w1 = max(tb, ta);
  }
  for (int e = tid; e < C::TAB_DOUBLES; e += C::NTHREADS) sTab[e] = g_ellip_tab[e];
  if (tid == 0) {
    for (int s = 0; s < NST; ++s) mbar_init(&full[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();

  // Tensor pairs of this thread: lane (gq, tq) of warp w evaluates (i = 8 iblk + gq, j = 4 k4 + tq) for the fragment
  // blocks blk = w + NWARPS u = iblk * 4 + k4 -- one warp store per component = 32 consecutive doubles (no conflicts).
  constexpr int NW = C::NTHREADS / 32, NU = C::PAIRS_PER_THREAD;
  double ri[NU], zi[NU];
  // NW is a multiple of 4, so every block of this thread has the same k4 = warp & 3: one source point per tile
  const int jl = (warp & 3) * 4 + tq;
  constexpr int CS = (C::TI / 8) * 4 * 32;
  PairEval pe[NU];
  auto store_tile = [&](int buf) {
    double* dst = sA + buf * C::A_DOUBLES + (warp << 5) + lane;
#pragma unroll
    for (int u = 0; u < NU; ++u) {
      const Tensor5 U = pe[u].finish();
      double* d = dst + ((NW * u) << 5);
      d[0] = U.UDrr;
      d[CS] = U.UDrz;
      d[2 * CS] = U.UDzz;
      d[3 * CS] = U.UKrr;
      d[4 * CS] = U.UKzr;
    }
  };

  double acc[WI_T][WC_T][5][2];
#pragma unroll
  for (int x = 0; x < WI_T; ++x)
#pragma unroll
    for (int n = 0; n < WC_T; ++n)
#pragma unroll
      for (int k = 0; k < 5; ++k) acc[x][n][k][0] = acc[x][n][k][1] = 0.0;

  unsigned cnt = 0;  // source-tile steps done by this CTA: stage = cnt % NST, mbarrier parity = (cnt / NST) & 1
  do {
  int it, ct, t0, nt, plane;
  bool whole;
  int rem_tile = -1;  // index of a partial-wave tile held in part
  if (stream_tiles) {
    int tile;
    if (seg_k < seg_q) {
      tile = seg_k * (int)gridDim.x + (int)blockIdx.x;
      ++seg_k;
      t0 = 0;
      nt = njt;
    } else {
      const int tr = (int)(w0 / njt);
      tile = seg_q * (int)gridDim.x + tr;
      t0 = (int)(w0 - (long long)tr * njt);
      nt = (int)min((long long)(njt - t0), w1 - w0);
      w0 += nt;
      if (nt < njt) rem_tile = tr;
    }
    ct = tile / stream_itiles;
    it = tile - ct * stream_itiles;
    plane = 0;
    whole = nt == njt;
  } else {
    it = blockIdx.x;
    ct = blockIdx.y;
    t0 = (int)w0;
    nt = (int)(w1 - w0);
    plane = blockIdx.z;
    whole = true;
    w0 += nt;
  }
  const int i0 = it * C::TI;
  const double* Fct = F + (long long)ct * njt * C::STAGE_DOUBLES;
  if (tid == 0) {
    for (int s = 0; s < NST && s < nt; ++s) {
      uint64_t* bar = &full[(cnt + s) % NST];
      mbar_expect_tx(bar, C::STAGE_DOUBLES * 8);
      bulk_g2s(sB + ((cnt + s) % NST) * C::STAGE_DOUBLES, Fct + (long long)(t0 + s) * C::STAGE_DOUBLES,
               C::STAGE_DOUBLES * 8, bar);
    }
  }
  // coordinates of the first two source tiles (later tiles arrive by cp.async two steps ahead of their use)
  if (tid < 4 * K2G_TJ && (tid >> 5) < nt) {
    const int tl = tid >> 5, e = tid & 31;
    const double* src = (e < K2G_TJ ? ip_r : ip_z) + j0 + (t0 + tl) * K2G_TJ + (e & (K2G_TJ - 1));
    sXY[tl * 2 * K2G_TJ + e] = *src;
  }
#pragma unroll
  for (int u = 0; u < NU; ++u) {
    const int ig = min(i0 + ((warp + NW * u) >> 2) * 8 + gq, n_i - 1);
    ri[u] = ip_r[ig];
    zi[u] = ip_z[ig];
  }
  __syncthreads();
  {
#pragma unroll
    for (int u = 0; u < NU; ++u) {
      pe[u].geometry(ri[u], zi[u], sXY[jl], sXY[K2G_TJ + jl], sTab);
      pe[u].template steps<LANDAU_ELLIP_TAB_DEG - 1, 0>();
    }
    store_tile(0);
  }
  __syncthreads();

  // Horner steps of the NEXT tile's tensor, cut in four and placed between the four k-blocks of DMMAs
  constexpr int D = LANDAU_ELLIP_TAB_DEG, H1 = D - 1 - D / 3, H2 = H1 - D / 3;
  for (int tt = 0; tt < nt; ++tt, ++cnt) {
    const int stage = cnt % NST;
    const bool more = tt + 1 < nt;
    mbar_wait(&full[stage], (cnt / NST) & 1);
    const double* A = sA + (tt & 1) * C::A_DOUBLES;
    const double* Bst = sB + stage * C::STAGE_DOUBLES;
    if (tt + 2 < nt && tid < K2G_TJ) {  // coordinates of the tile after next: 16 x 16 bytes, landed by the end of the step
      const int e = tid * 2;        // doubles 0..15 = r, 16..31 = z
      const double* src = (e < K2G_TJ ? ip_r : ip_z) + j0 + (t0 + tt + 2) * K2G_TJ + (e & (K2G_TJ - 1));
      cp_async16(sXY + ((tt + 2) & 3) * 2 * K2G_TJ + e, src);
    }
    cp_async_commit();
    if (more) {
      const double* xy = sXY + ((tt + 1) & 3) * 2 * K2G_TJ;
      const double rj = xy[jl], zj = xy[K2G_TJ + jl];
#pragma unroll
      for (int u = 0; u < NU; ++u) pe[u].geometry(ri[u], zi[u], rj, zj, sTab);
    }
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) {
      double a[WI_T][5];
#pragma unroll
      for (int x = 0; x < WI_T; ++x)
#pragma unroll
        for (int k = 0; k < 5; ++k) a[x][k] = A[k * CS + (((wi * WI_T + x) * 4 + ks) << 5) + lane];
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
      if (more) {
#pragma unroll
        for (int u = 0; u < NU; ++u) {
          if (ks == 0) pe[u].template steps<D - 1, H1 + 1>();
          if (ks == 1) pe[u].template steps<H1, H2 + 1>();
          if (ks == 2) pe[u].template steps<H2, 0>();
        }
        if (ks == 3) store_tile((tt + 1) & 1);
      }
    }
    cp_async_wait<0>();
    __syncthreads();
    if (tid == 0 && tt + NST < nt) {
      mbar_expect_tx(&full[stage], C::STAGE_DOUBLES * 8);
      bulk_g2s(sB + stage * C::STAGE_DOUBLES, Fct + (long long)(t0 + tt + NST) * C::STAGE_DOUBLES, C::STAGE_DOUBLES * 8,
               &full[stage]);
    }
  }

  if (!whole) {
    // Partial tile: parts are numbered by CTA.  first = lowest CTA whose share [lo(p), lo(p+1)) of the partial wave
    // meets this tile, lo(p) = floor(R p / P).
    const long long R = (long long)(stream_tiles - seg_q * (int)gridDim.x) * njt, P = gridDim.x;
    const long long tb = (long long)rem_tile * njt, te = tb + njt;
    int first = (int)(tb * P / R);
    while (first > 0 && R * first / P > tb) --first;
    while (R * (first + 1) / P <= tb) ++first;
    int lastp = (int)((te - 1) * P / R);
    while (lastp + 1 < (int)P && R * (lastp + 1) / P < te) ++lastp;
    while (R * lastp / P >= te) --lastp;
    const int nparts = lastp - first + 1, mypart = (int)blockIdx.x - first;
    double* mine = part_buf + ((long long)rem_tile * part_stride + mypart) * (C::ACC_PER_THREAD * C::NTHREADS) + tid;
    {
      int e = 0;
#pragma unroll
      for (int x = 0; x < WI_T; ++x)
#pragma unroll
        for (int n = 0; n < WC_T; ++n)
#pragma unroll
          for (int k = 0; k < 5; ++k)
#pragma unroll
            for (int h = 0; h < 2; ++h, ++e) mine[e * C::NTHREADS] = acc[x][n][k][h];
    }
    __threadfence();
    __syncthreads();
    __shared__ int s_last;
    if (tid == 0) s_last = atomicAdd(part_count + rem_tile, 1) == nparts - 1;
    __syncthreads();
    whole = s_last;
    if (whole) {  // every part is visible: add them in part order
      __threadfence();
      const double* src = part_buf + (long long)rem_tile * part_stride * (C::ACC_PER_THREAD * C::NTHREADS) + tid;
      int e = 0;
#pragma unroll
      for (int x = 0; x < WI_T; ++x)
#pragma unroll
        for (int n = 0; n < WC_T; ++n)
#pragma unroll
          for (int k = 0; k < 5; ++k)
#pragma unroll
            for (int h = 0; h < 2; ++h, ++e) {
              double sum = 0.0;
              for (int q = 0; q < nparts; ++q) sum += __ldcg(src + ((long long)q * C::ACC_PER_THREAD + e) * C::NTHREADS);
              acc[x][n][k][h] = sum;
            }
    }
  }
  // C fragment: row gq (field point), columns 2 tq, 2 tq + 1
#pragma unroll
  for (int x = 0; x < WI_T; ++x) {
    const int i = i0 + (wi * WI_T + x) * 8 + gq;
#pragma unroll
    for (int n = 0; n < WC_T; ++n)
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int col = ct * C::TC + (wc * WC_T + n) * 8 + 2 * tq + h;
        if (whole && i < n_i && col < ncols) {
          double* dst = G + plane * g_split_stride + ((long long)(gcol0 + col) * 5) * n_i + i;
#pragma unroll
          for (int k = 0; k < 5; ++k) dst[(long long)k * n_i] = acc[x][n][k][h];
        }
#pragma unroll
        for (int k = 0; k < 5; ++k) acc[x][n][k][h] = 0.0;
      }
  }
  } while (seg_k < seg_q || w0 < w1);  // segments (an empty j-split still stores its zeros)
}

}  // namespace landau
