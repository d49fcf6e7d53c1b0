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

template <int NT>
__global__ void __launch_bounds__(K2D_WARPS * 32) k3v_inner_dmma(const double* __restrict__ px, const double* __restrict__ py,
                                                                const double* __restrict__ pz, int n_pad, Ranges3 rg, int nbc,
                                                                int nsplit, const double* __restrict__ F, double* __restrict__ G,
                                                                long long split_stride) {
  constexpr int NCOL = 8 * NT;
  __shared__ double sF[NCOL * 4 * K2D_LD], sxyz[3][K2D_TJ];
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
  for (int jt = ta; jt < tb; ++jt) {
    const int j0 = jt * K2D_TJ;
    __syncthreads();
    if (tid < 3 * K2D_TJ) sxyz[tid / K2D_TJ][tid % K2D_TJ] = (tid < K2D_TJ ? px : tid < 2 * K2D_TJ ? py : pz)[j0 + tid % K2D_TJ];
    for (int e = tid; e < NCOL * 4 * K2D_TJ; e += K2D_WARPS * 32) {
      const int row = e / K2D_TJ, j = e % K2D_TJ;  // row = col * 4 + comp
      sF[row * K2D_LD + j] = bfirst + row / 4 < nbc ? Fc[(long long)row * n_pad + j0 + j] : 0.0;
    }
    __syncthreads();
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) {
      const int j = ks * 4 + t;
      const Tensor6 U = landau_tensor_3v(xi, yi, zi, ri2, sxyz[0][j], sxyz[1][j], sxyz[2][j]);
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

// returns 0 or a landau_status; *nsplit_out = parts the source range was cut into (K2b adds them)
inline int launch_inner_dmma(const double* px, const double* py, const double* pz, int n_pad, const Ranges3& rg, int n_classes,
                             int nbc, int nsplit, const double* F, double* G, long long split_stride, cudaStream_t st) {
  const int nt = nbc > 16 ? 4 : nbc > 8 ? 2 : 1, ncol = 8 * nt;
  const dim3 grid(n_pad / (K2D_WARPS * 8), n_classes * ((nbc + ncol - 1) / ncol), nsplit);
  if (nt == 4)
    k3v_inner_dmma<4><<<grid, K2D_WARPS * 32, 0, st>>>(px, py, pz, n_pad, rg, nbc, nsplit, F, G, split_stride);
  else if (nt == 2)
    k3v_inner_dmma<2><<<grid, K2D_WARPS * 32, 0, st>>>(px, py, pz, n_pad, rg, nbc, nsplit, F, G, split_stride);
  else
    k3v_inner_dmma<1><<<grid, K2D_WARPS * 32, 0, st>>>(px, py, pz, n_pad, rg, nbc, nsplit, F, G, split_stride);
  return 0;
}

}  // namespace landau3v
