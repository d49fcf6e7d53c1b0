// landau3v_dmma.cuh -- K2 of the 3V variant on the FP64 MMA pipe.
//
// With the tensor shared by all source columns, a2 is the dense FP64 contraction  G_k[i, c] += U_k(i, j) F_l[j, c]  over
// the source points j (15 products per (i, j, column): 6 for G^D = U f, 9 for G^K = U . grad f) whose A operand is generated
// on the fly.  It is issued as mma.sync.m8n8k4.f64 (SASS DMMA; tcgen05 has no FP64 kind): a warp owns 8 field points, lane
// (g, t) evaluates the tensor of ONE pair (field point g, source point t of the current four) -- 32 distinct pairs per
// warp and k-step, nothing evaluated twice -- and that value is the A fragment of the DMMAs against the F fragments of up
// to NT x 8 columns.  The 3-D tensor costs ~25 FP64 instructions per pair against 15 NT DMMAs (= 120 NT scalar-FMA slots per
// lane), so the kernel sits nearer the DMMA peak than its 2V counterpart (~140 FLOP of elliptic-integral work per pair).
// A CTA is 4 warps (32 field points) sharing one shared-memory F tile of 16 source points.  Two launch modes: persistent CTAs
// sharing all (item, source tile) steps evenly (stream mode, the default), or a grid whose source range is cut into `nsplit`
// parts (grid z) when the tiles alone do not fill the machine, the parts being added by K2b (first version, kept for A/B).
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

// One segment of work: the CTA's 32 field points of field tile `ft`, columns bfirst .. of class `cls`, source tiles ta .. tb - 1,
// added to acc.  stage: two shared-memory tiles (F rows, then x, y, z), rows past `nrows` are kept at zero.
template <int NT>
__device__ __forceinline__ void inner_dmma_segment(const double* __restrict__ px, const double* __restrict__ py,
                                                   const double* __restrict__ pz, int n_pad, int nbc, const double* __restrict__ F,
                                                   int ft, int cls, int bfirst, int ta, int tb, double (&acc)[NT][9][2],
                                                   double* stage0) {
  constexpr int NCOL = 8 * NT, TILE = NCOL * 4 * K2D_LD + 3 * K2D_TJ;  // doubles per stage
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, g = lane >> 2, t = lane & 3;
  const int i = ft * (K2D_WARPS * 8) + warp * 8 + g;
  const double xi = px[i], yi = py[i], zi = pz[i];
  const double ri2 = fma(xi, xi, fma(yi, yi, zi * zi));
  const double* Fc = F + ((long long)cls * nbc + bfirst) * 4 * n_pad;
  const int nrows = min(NCOL, nbc - bfirst) * 4;  // rows (column, component) that exist; the others stay zero
  // a source tile travels global -> shared memory by 8-byte async copies, one tile ahead of its use
  auto fetch = [&](int jt) {
    double* st = stage0 + (jt & 1) * TILE;
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
    const double* sF = stage0 + (jt & 1) * TILE;
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
}

// C fragment: lane (g, t) holds field point g, columns 2 t and 2 t + 1 of every n-tile
template <int NT>
__device__ __forceinline__ void inner_dmma_store(double* __restrict__ Gs, int n_pad, int nbc, int ft, int cls, int bfirst,
                                                 const double (&acc)[NT][9][2]) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, g = lane >> 2, t = lane & 3;
  const int i = ft * (K2D_WARPS * 8) + warp * 8 + g;
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

// grid mode: one CTA per (field tile, class x column tile, part of the source range); the parts are planes of G added by K2b
template <int NT>
__global__ void __launch_bounds__(K2D_WARPS * 32) k3v_inner_dmma(const double* __restrict__ px, const double* __restrict__ py,
                                                                const double* __restrict__ pz, int n_pad, Ranges3 rg, int nbc,
                                                                int nsplit, const double* __restrict__ F, double* __restrict__ G,
                                                                long long split_stride) {
  constexpr int NCOL = 8 * NT, TILE = NCOL * 4 * K2D_LD + 3 * K2D_TJ;
  __shared__ double stage[2 * TILE];
  const int tiles_per_class = (nbc + NCOL - 1) / NCOL;
  const int cls = blockIdx.y / tiles_per_class, bfirst = (blockIdx.y % tiles_per_class) * NCOL;
  double acc[NT][9][2];
#pragma unroll
  for (int n = 0; n < NT; ++n)
#pragma unroll
    for (int k = 0; k < 9; ++k) acc[n][k][0] = acc[n][k][1] = 0.0;
  // this CTA's part of the class's source range, in tiles
  const int t0 = rg.j0[cls] / K2D_TJ, t1 = rg.j1[cls] / K2D_TJ;
  const int ta = t0 + (int)((long long)(t1 - t0) * blockIdx.z / nsplit), tb = t0 + (int)((long long)(t1 - t0) * (blockIdx.z + 1) / nsplit);
  for (int e = threadIdx.x; e < 2 * TILE; e += K2D_WARPS * 32) stage[e] = 0.0;
  __syncthreads();
  inner_dmma_segment<NT>(px, py, pz, n_pad, nbc, F, blockIdx.x, cls, bfirst, ta, tb, acc, stage);
  inner_dmma_store<NT>(G + (long long)blockIdx.z * split_stride, n_pad, nbc, blockIdx.x, cls, bfirst, acc);
}

// Work layout of the stream mode: items = (class, column tile, field tile), field tile fastest; item (c, ., .) has
// njt[c] source-tile steps; steps are numbered item by item.
struct StreamPlan3 {
  int n_ft, col_tiles, n_classes;
  int njt[MAX_TERMS];
  long long step0[MAX_TERMS + 1];  // first step of every class
};

// stream mode: P persistent CTAs share the W = sum of steps evenly, CTA p takes steps [W p / P, W (p + 1) / P) -- whole items
// and at most one cut item at either end.  The part of a cut item goes to part_buf (slot 2 p: the CTA begins inside the
// item, 2 p + 1: it began in an earlier one); the CTA that arrives last at the item's counter adds the parts in CTA order and
// stores the item: deterministic, no atomics on G, one plane.  Needs W >= P (no CTA without work).
template <int NT>
__global__ void __launch_bounds__(K2D_WARPS * 32) k3v_inner_dmma_stream(const double* __restrict__ px, const double* __restrict__ py,
                                                                       const double* __restrict__ pz, int n_pad, Ranges3 rg, int nbc,
                                                                       StreamPlan3 pl, const double* __restrict__ F,
                                                                       double* __restrict__ G, double* __restrict__ part_buf,
                                                                       int* __restrict__ part_count) {
  constexpr int NCOL = 8 * NT, TILE = NCOL * 4 * K2D_LD + 3 * K2D_TJ, ACC = NT * 18;
  __shared__ double stage[2 * TILE];
  __shared__ int s_last;
  const int tid = threadIdx.x;
  const long long W = pl.step0[pl.n_classes], P = gridDim.x;
  long long w = W * blockIdx.x / P;
  const long long w_end = W * (blockIdx.x + 1) / P, w_begin = w;
  auto cta_of = [&](long long step) { return (int)(((step + 1) * P - 1) / W); };  // the CTA whose share holds `step`
  double acc[NT][9][2];
  while (w < w_end) {
    int cls = 0;
    while (cls + 1 < pl.n_classes && w >= pl.step0[cls + 1]) ++cls;
    const int njt = pl.njt[cls];
    const long long rel = w - pl.step0[cls];
    const int item_in_class = (int)(rel / njt), t_first = (int)(rel - (long long)item_in_class * njt);
    const int nt = (int)min((long long)(njt - t_first), w_end - w);
    const int ct = item_in_class / pl.n_ft, ft = item_in_class - ct * pl.n_ft, bfirst = ct * NCOL;
    const int item = cls * pl.col_tiles * pl.n_ft + item_in_class;
#pragma unroll
    for (int n = 0; n < NT; ++n)
#pragma unroll
      for (int k = 0; k < 9; ++k) acc[n][k][0] = acc[n][k][1] = 0.0;
    __syncthreads();  // the stage of the previous segment is no longer read
    for (int e = tid; e < 2 * TILE; e += K2D_WARPS * 32) stage[e] = 0.0;
    __syncthreads();
    const int tbase = rg.j0[cls] / K2D_TJ;
    inner_dmma_segment<NT>(px, py, pz, n_pad, nbc, F, ft, cls, bfirst, tbase + t_first, tbase + t_first + nt, acc, stage);
    bool store = true;
    if (nt < njt) {  // cut item
      const long long a = w - t_first, b = a + njt;  // the item's steps
      const int first = cta_of(a), last = cta_of(b - 1), nparts = last - first + 1;
      double* mine = part_buf + ((long long)(2 * blockIdx.x + (w_begin < a ? 1 : 0)) * ACC) * (K2D_WARPS * 32) + tid;
      {
        int e = 0;
#pragma unroll
        for (int n = 0; n < NT; ++n)
#pragma unroll
          for (int k = 0; k < 9; ++k)
#pragma unroll
            for (int h = 0; h < 2; ++h, ++e) mine[e * (K2D_WARPS * 32)] = acc[n][k][h];
      }
      __threadfence();
      __syncthreads();
      if (tid == 0) s_last = atomicAdd(part_count + item, 1) == nparts - 1;
      __syncthreads();
      store = s_last;
      if (store) {  // every part is visible: add them in CTA order
        __threadfence();
#pragma unroll
        for (int n = 0; n < NT; ++n)
#pragma unroll
          for (int k = 0; k < 9; ++k) acc[n][k][0] = acc[n][k][1] = 0.0;
        for (int q = 0; q < nparts; ++q) {
          const int c = first + q;
          const long long c_begin = W * c / P;
          const double* src = part_buf + ((long long)(2 * c + (c_begin < a ? 1 : 0)) * ACC) * (K2D_WARPS * 32) + tid;
          int e = 0;
#pragma unroll
          for (int n = 0; n < NT; ++n)
#pragma unroll
            for (int k = 0; k < 9; ++k)
#pragma unroll
              for (int h = 0; h < 2; ++h, ++e) acc[n][k][h] += __ldcg(src + e * (K2D_WARPS * 32));
        }
      }
    }
    if (store) inner_dmma_store<NT>(G, n_pad, nbc, ft, cls, bfirst, acc);
    w += nt;
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

// stream mode: occupancy, scratch need (doubles: two accumulator slots per CTA + one counter per item) and launch
template <int NT>
inline int inner_dmma_stream_ctas_per_sm_t() {
  int n = 0;
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k3v_inner_dmma_stream<NT>, K2D_WARPS * 32, 0);
  return n > 0 ? n : 1;
}
inline int inner_dmma_stream_ctas_per_sm(int nt) {
  return nt == 4 ? inner_dmma_stream_ctas_per_sm_t<4>() : nt == 2 ? inner_dmma_stream_ctas_per_sm_t<2>() : inner_dmma_stream_ctas_per_sm_t<1>();
}
inline StreamPlan3 inner_dmma_stream_plan(int n_pad, const Ranges3& rg, int n_classes, int nbc) {
  StreamPlan3 pl;
  const int ncol = 8 * inner_dmma_nt(nbc);
  pl.n_ft = n_pad / (K2D_WARPS * 8);
  pl.col_tiles = (nbc + ncol - 1) / ncol;
  pl.n_classes = n_classes;
  pl.step0[0] = 0;
  for (int c = 0; c < n_classes; ++c) {
    pl.njt[c] = (rg.j1[c] - rg.j0[c]) / K2D_TJ;
    pl.step0[c + 1] = pl.step0[c] + (long long)pl.njt[c] * pl.col_tiles * pl.n_ft;
  }
  return pl;
}
inline size_t inner_dmma_stream_scratch(int nt, int n_ctas, const StreamPlan3& pl) {
  return (size_t)2 * n_ctas * nt * 18 * (K2D_WARPS * 32) + ((size_t)pl.n_classes * pl.col_tiles * pl.n_ft + 1) / 2 + 1;
}
inline int launch_inner_dmma_stream(const double* px, const double* py, const double* pz, int n_pad, const Ranges3& rg, int nbc,
                                    const StreamPlan3& pl, int n_ctas, const double* F, double* G, double* scratch, cudaStream_t st) {
  const int nt = inner_dmma_nt(nbc);
  const size_t acc_doubles = (size_t)2 * n_ctas * nt * 18 * (K2D_WARPS * 32);
  int* count = reinterpret_cast<int*>(scratch + acc_doubles);
  if (cudaMemsetAsync(count, 0, sizeof(int) * pl.n_classes * pl.col_tiles * pl.n_ft, st) != cudaSuccess) return -1;
  if (nt == 4)
    k3v_inner_dmma_stream<4><<<n_ctas, K2D_WARPS * 32, 0, st>>>(px, py, pz, n_pad, rg, nbc, pl, F, G, scratch, count);
  else if (nt == 2)
    k3v_inner_dmma_stream<2><<<n_ctas, K2D_WARPS * 32, 0, st>>>(px, py, pz, n_pad, rg, nbc, pl, F, G, scratch, count);
  else
    k3v_inner_dmma_stream<1><<<n_ctas, K2D_WARPS * 32, 0, st>>>(px, py, pz, n_pad, rg, nbc, pl, F, G, scratch, count);
  return 0;
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
