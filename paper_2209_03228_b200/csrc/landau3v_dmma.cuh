// landau3v_dmma.cuh -- K2 of the 3V variant on the FP64 MMA pipe.
//
// With the tensor shared by all source columns, a2 is the dense FP64 contraction  G_k[i, c] += U_k(i, j) F_l[j, c]  over
// the source points j (15 products per (i, j, column): 6 for G^D = U f, 9 for G^K = U . grad f) whose A operand is generated
// on the fly.  It is issued as mma.sync.m8n8k4.f64 (SASS DMMA; tcgen05 has no FP64 kind): a warp owns 8 field points, lane
// (g, t) evaluates the tensor of ONE pair (field point g, source point t of the current four) -- 32 distinct pairs per
// warp and k-step, nothing evaluated twice -- and that value is the A fragment of the DMMAs against the F fragments of up
// to NT x 8 columns.  The 3-D tensor costs ~25 FP64 instructions per pair against 15 NT DMMAs (= 120 NT scalar-FMA slots per
// lane), so the kernel sits nearer the DMMA peak than its 2V counterpart (~140 FLOP of elliptic-integral work per pair).
// A CTA is 4 warps (32 field points) sharing one shared-memory F tile of 16 source points; the source range is cut into
// `nsplit` parts (grid z) when the tiles alone do not fill the machine, the parts are added by K2b.
#pragma once
#include "landau3v_kernels.cuh"

namespace landau3v {

constexpr int K2D_TJ = 16;  // source points per shared-memory tile (four k-steps)
constexpr int K2D_LD = 17;  // row stride of the F tile: lanes (g, t) of a half-warp hit 16 distinct banks
constexpr int K2D_WARPS = 4;

__device__ __forceinline__ void dmma3(double& d0, double& d1, double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

__device__ __forceinline__ void cp8_3v(double* smem, const double* gmem) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem));
}

template <int NT>
__global__ void __launch_bounds__(K2D_WARPS * 32) k3v_inner_dmma(const double* __restrict__ px, const double* __restrict__ py,
                                                                const double* __restrict__ pz, int n_pad, Ranges3 rg, int nbc,
                                                                int nsplit, const double* __restrict__ F, double* __restrict__ G,
                                                                long long split_stride) {
  constexpr int NCOL = 8 * NT, TILE = NCOL * 4 * K2D_LD + 3 * K2D_TJ;  // doubles per stage: F rows, then x, y, z
  __shared__ double stage[2][TILE];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, t = lane & 3;
  const int tiles_per_class = (nbc + NCOL - 1) / NCOL;
  const int cls = blockIdx.y / tiles_per_class, bfirst = (blockIdx.y % tiles_per_class) * NCOL;
  const int i = blockIdx.x * (K2D_WARPS * 8) + warp * 8 + g;
  const double xi = px[i], yi = py[i], zi = pz[i];
  const double ri2 = fma(xi, xi, fma(yi, yi, zi * zi));
  double acc[NT][9][2];
#pragma unroll
  for (int n = 0; n < NT; ++n)
#pragma unroll
    for (int k = 0; k < 9; ++k) acc[n][k][0] = acc[n][k][1] = 0.0;
  // this CTA's part of the class's source range, in tiles
  const int t0 = rg.j0[cls] / K2D_TJ, t1 = rg.j1[cls] / K2D_TJ;
  const int ta = t0 + (int)((long long)(t1 - t0) * blockIdx.z / nsplit), tb = t0 + (int)((long long)(t1 - t0) * (blockIdx.z + 1) / nsplit);
  const double* Fc = F + ((long long)cls * nbc + bfirst) * 4 * n_pad;
  const int nrows = min(NCOL, nbc - bfirst) * 4;  // rows (column, component) that exist; the others stay zero
  for (int e = tid; e < 2 * TILE; e += K2D_WARPS * 32) (&stage[0][0])[e] = 0.0;
  __syncthreads();
  // a source tile travels global -> shared memory by 8-byte async copies, one tile ahead of its use
  auto fetch = [&](int jt) {
    double* st = stage[jt & 1];
    const int j0 = jt * K2D_TJ;
    for (int e = tid; e < nrows * K2D_TJ; e += K2D_WARPS * 32) {
      const int row = e / K2D_TJ, j = e % K2D_TJ;
      cp8_3v(st + row * K2D_LD + j, Fc + (long long)row * n_pad + j0 + j);
    }
    if (tid < 3 * K2D_TJ) cp8_3v(st + NCOL * 4 * K2D_LD + tid, (tid < K2D_TJ ? px : tid < 2 * K2D_TJ ? py : pz) + j0 + tid % K2D_TJ);
  };
  if (ta < tb) fetch(ta);
  asm volatile("cp.async.commit_group;");
  for (int jt = ta; jt < tb; ++jt) {
    asm volatile("cp.async.wait_group 0;");
    __syncthreads();  // tile jt has landed for everybody, and everybody has finished tile jt - 1 (whose buffer is refilled now)
    if (jt + 1 < tb) fetch(jt + 1);
    asm volatile("cp.async.commit_group;");
    const double* sF = stage[jt & 1];
    const double* sxyz = sF + NCOL * 4 * K2D_LD;
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) {
      const int j = ks * 4 + t;
      const Tensor6 U = landau_tensor_3v(xi, yi, zi, ri2, sxyz[j], sxyz[K2D_TJ + j], sxyz[2 * K2D_TJ + j]);
#pragma unroll
      for (int n = 0; n < NT; ++n) {
        const double* fr = sF + (n * 8 + g) * 4 * K2D_LD + j;
        const double f = fr[0], gx = fr[K2D_LD], gy = fr[2 * K2D_LD], gz = fr[3 * K2D_LD];
        dmma3(acc[n][0][0], acc[n][0][1], U.xx, f);
        dmma3(acc[n][1][0], acc[n][1][1], U.xy, f);
        dmma3(acc[n][2][0], acc[n][2][1], U.xz, f);
        dmma3(acc[n][3][0], acc[n][3][1], U.yy, f);
        dmma3(acc[n][4][0], acc[n][4][1], U.yz, f);
        dmma3(acc[n][5][0], acc[n][5][1], U.zz, f);
        dmma3(acc[n][6][0], acc[n][6][1], U.xx, gx);
        dmma3(acc[n][7][0], acc[n][7][1], U.xy, gx);
        dmma3(acc[n][8][0], acc[n][8][1], U.xz, gx);
        dmma3(acc[n][6][0], acc[n][6][1], U.xy, gy);
        dmma3(acc[n][7][0], acc[n][7][1], U.yy, gy);
        dmma3(acc[n][8][0], acc[n][8][1], U.yz, gy);
        dmma3(acc[n][6][0], acc[n][6][1], U.xz, gz);
        dmma3(acc[n][7][0], acc[n][7][1], U.yz, gz);
        dmma3(acc[n][8][0], acc[n][8][1], U.zz, gz);
      }
    }
  }
  // C fragment: lane (g, t) holds field point g, columns 2 t and 2 t + 1 of every n-tile
  double* Gs = G + (long long)blockIdx.z * split_stride;
#pragma unroll
  for (int n = 0; n < NT; ++n)
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const int col = bfirst + n * 8 + 2 * t + h;
      if (col < nbc) {
        double* dst = Gs + ((long long)cls * nbc + col) * 9 * n_pad + i;
#pragma unroll
        for (int k = 0; k < 9; ++k) dst[(long long)k * n_pad] = acc[n][k][h];
      }
    }
}

template <int NT>
inline void launch_inner_dmma_t(const double* px, const double* py, const double* pz, int n_pad, const Ranges3& rg, int n_classes,
                                int nbc, int nsplit, const double* F, double* G, long long split_stride, cudaStream_t st) {
  const dim3 grid(n_pad / (K2D_WARPS * 8), n_classes * ((nbc + 8 * NT - 1) / (8 * NT)), nsplit);
  k3v_inner_dmma<NT><<<grid, K2D_WARPS * 32, 0, st>>>(px, py, pz, n_pad, rg, nbc, nsplit, F, G, split_stride);
}
inline int inner_dmma_nt(int nbc) { return nbc > 16 ? 4 : nbc > 8 ? 2 : 1; }

// CTAs of the variant that fit on one SM (registers / shared memory), queried once per variant
inline int inner_dmma_ctas_per_sm(int nt) {
  int n = 0;
  if (nt == 4)
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k3v_inner_dmma<4>, K2D_WARPS * 32, 0);
  else if (nt == 2)
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k3v_inner_dmma<2>, K2D_WARPS * 32, 0);
  else
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k3v_inner_dmma<1>, K2D_WARPS * 32, 0);
  return n > 0 ? n : 1;
}

// Parts to cut the source range into: the smallest count for which the CTAs fill at least 95 % of the waves they take
// (304 field tiles on 148 x 2 slots are 1.03 waves and would take the time of 2), else the best one found.
inline int inner_dmma_split(long long items, long long slots, int max_split) {
  int best = 1;
  double best_eff = 0.0;
  for (int n = 1; n <= max_split; ++n) {
    const long long ctas = items * n, waves = (ctas + slots - 1) / slots;
    const double eff = (double)ctas / (double)(waves * slots);
    if (eff > best_eff + 1e-9) {
      best_eff = eff;
      best = n;
    }
    if (eff >= 0.95) return n;
  }
  return best;
}

inline int launch_inner_dmma(const double* px, const double* py, const double* pz, int n_pad, const Ranges3& rg, int n_classes,
                             int nbc, int nsplit, const double* F, double* G, long long split_stride, cudaStream_t st) {
  const int nt = inner_dmma_nt(nbc);
  if (nt == 4)
    launch_inner_dmma_t<4>(px, py, pz, n_pad, rg, n_classes, nbc, nsplit, F, G, split_stride, st);
  else if (nt == 2)
    launch_inner_dmma_t<2>(px, py, pz, n_pad, rg, n_classes, nbc, nsplit, F, G, split_stride, st);
  else
    launch_inner_dmma_t<1>(px, py, pz, n_pad, rg, n_classes, nbc, nsplit, F, G, split_stride, st);
  return 0;
}

}  // namespace landau3v
