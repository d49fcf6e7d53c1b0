// landau_kernels.cuh -- device code of the batched Landau Jacobian path (sm_100a).
//
//   K1  k1_fields        a1: source fields  F = w_j * (sum over species) {f, df/dr, df/dz} at the IPs
//   K2  k2_inner_dfma    a2: inner integral, plain FP64 FMA version (few columns)
//       k2_inner_dmma    a2: inner integral on the DMMA pipe, tensor generated per warp (8 .. 96 columns)
//       k2_inner_gemm    a2: (k2_gemm.cuh) tensor tile shared by the CTA, TMA-staged source tiles (many columns)
//   K2b k2b_combine      a2: D_a, K_a = species combination of the partial sums (also sums the j-splits)
//   K3  k3_ring          a3+a4: (k3_ring.cuh) DMMA element matrices in a shared-memory ring, gathered into batched CSR
//       k3_elem_matrix, k3_gather   a3+a4 without a ring schedule (triangles, ...): element matrices to scratch, slot gather
//       k3_assemble      a3+a4: first version, one thread per CSR slot integrating its own entries (kept for A/B)
//   K3' k3_elem_apply_all, k3_apply_gather_all   a5: operator application, one launch pair for all species
//   K4  k4_tfqmr         (k4_solve.cuh) batched TFQMR + Jacobi solve, the step after the path
//
// Notation follows PAPER.md sec. 2 and DESIGN.md: i = field point, j = source point, U^D / U^K the gyro-averaged
// Landau tensor contracted with the field / source unit vectors.
#pragma once
#include <cuda_runtime.h>

#include "ellip_coeffs.h"

namespace landau {

// ------------------------------------------------------------------------------------------------------------
// Elliptic pieces.  Coefficients are compile-time constants: every Horner step is a DFMA with an immediate / uniform-
// register operand that the assembler rematerialises where needed (no loads, nothing to hoist out of the tile loops
// and spill -- __constant__ tables were hoisted by the compiler into registers and from there into local memory).
// ------------------------------------------------------------------------------------------------------------
static constexpr double c_L_A_E[] = LANDAU_ELLIP_L_A_E_COEFFS;
static constexpr double c_L_B_E[] = LANDAU_ELLIP_L_B_E_COEFFS;
static constexpr double c_L_A_DC[] = LANDAU_ELLIP_L_A_DC_COEFFS;
static constexpr double c_L_B_DC[] = LANDAU_ELLIP_L_B_DC_COEFFS;
static constexpr double c_L_A_Q[] = LANDAU_ELLIP_L_A_Q_COEFFS;
static constexpr double c_L_B_Q[] = LANDAU_ELLIP_L_B_Q_COEFFS;

template <const double* C, int N>
struct HornerStep {
  static __device__ __forceinline__ double run(double acc, double t) {
    constexpr double c = C[N];
    return HornerStep<C, N - 1>::run(fma(acc, t, c), t);
  }
};
template <const double* C>
struct HornerStep<C, -1> {
  static __device__ __forceinline__ double run(double acc, double) { return acc; }
};
template <const double* C, int DEG>
__device__ __forceinline__ double horner(double t) {
  constexpr double top = C[DEG];
  return HornerStep<C, DEG - 1>::run(top, t);
}

// (E, Dc, Q) at complement x = m' = 1 - m (given directly, never formed by subtraction), E = m' P0:
//   Dc = (K-E)/m,  Q = ((2-m)K - 2E)/m^2   -- see gen_ellip_coeffs.py.
// x >= 2^-TAB_BINADES (all but near-coincident pairs): table T.  The interval index is the exponent and the top two
// mantissa bits of x, the interval centre is x with the lower mantissa bits replaced by 100..0, so t = x - centre is
// exact; three degree-TAB_DEG Horner chains share the loads of one table row (L1-resident, 13 KB).  No branch on m,
// no logarithm: 3 (TAB_DEG) DFMA instead of 73 (old small-m fit) or ~140 (logarithmic form).
// x < 2^-TAB_BINADES: f = A_f(x) + ln(1/x) B_f(x) (fits valid for x < 1 - M_SPLIT).
__device__ __align__(16) const double g_ellip_tab[] = LANDAU_ELLIP_TAB_COEFFS;
constexpr double ELLIP_TAB_XMIN = 1.0 / (1 << LANDAU_ELLIP_TAB_BINADES);

// logarithmic form, x < 1 - M_SPLIT
__device__ __forceinline__ void ellip_pieces_log(double x, double& E, double& Dc, double& Q) {
  const double t = x - 0.5 * (1.0 - LANDAU_ELLIP_M_SPLIT);
  const double lg = -log(x);
  E = fma(lg, horner<c_L_B_E, LANDAU_ELLIP_L_B_E_DEG>(t), horner<c_L_A_E, LANDAU_ELLIP_L_A_E_DEG>(t));
  Dc = fma(lg, horner<c_L_B_DC, LANDAU_ELLIP_L_B_DC_DEG>(t), horner<c_L_A_DC, LANDAU_ELLIP_L_A_DC_DEG>(t));
  Q = fma(lg, horner<c_L_B_Q, LANDAU_ELLIP_L_B_Q_DEG>(t), horner<c_L_A_Q, LANDAU_ELLIP_L_A_Q_DEG>(t));
}

// Table evaluation in stages, so that a kernel can interleave the Horner steps with other work:
//   start(x) -> steps<HI, LO>() ... -> E, Dc, Q valid after steps down to 0 (x >= ELLIP_TAB_XMIN; smaller x index the
//   first interval and must be redone with ellip_pieces_log).
struct EllipTable {
  double t, E, Dc, Q;
  const double* row;
  __device__ __forceinline__ void start(double x, const double* __restrict__ tab) {
    constexpr int BIAS = (1023 - LANDAU_ELLIP_TAB_BINADES) << 2, D = LANDAU_ELLIP_TAB_DEG;
    const int idx = max(min((__double2hiint(x) >> 18) - BIAS, 4 * LANDAU_ELLIP_TAB_BINADES - 1), 0);  // x == 1: last
    t = x - __hiloint2double(((idx + BIAS) << 18) | 0x20000, 0);
    row = tab + idx * (D + 1) * 4;
    const double2 ed = *reinterpret_cast<const double2*>(row + 4 * D);
    E = ed.x;
    Dc = ed.y;
    Q = row[4 * D + 2];
  }
  template <int HI, int LO>
  __device__ __forceinline__ void steps() {
#pragma unroll
    for (int n = HI; n >= LO; --n) {
      const double2 ed = *reinterpret_cast<const double2*>(row + 4 * n);
      const double q = row[4 * n + 2];
      E = fma(E, t, ed.x);
      Dc = fma(Dc, t, ed.y);
      Q = fma(Q, t, q);
    }
  }
};

__device__ __forceinline__ void ellip_pieces(double x, double& E, double& Dc, double& Q) {
  if (x >= ELLIP_TAB_XMIN) {
    EllipTable e;
    e.start(x, g_ellip_tab);
    e.template steps<LANDAU_ELLIP_TAB_DEG - 1, 0>();
    E = e.E;
    Dc = e.Dc;
    Q = e.Q;
  } else {
    ellip_pieces_log(x, E, Dc, Q);
  }
}

// ------------------------------------------------------------------------------------------------------------
// 2V Landau tensor for the pair (field point (r,z), source point (rb,zb)); DESIGN.md "tensor":
//   s+- = (r +- rb)^2 + dz^2, m = 4 r rb / s+, m' = s-/s+, c = 4 / s+^{3/2}
//   UD_rr = c (4 rb^2 Q + dz^2 P0)         UK_rr = c (4 r rb Q + dz^2 m P2),  m P2 = m (P0 - Dc - Q)
//   UD_zz = c ((r-rb)^2 P0 + 4 r rb Dc)    UK_zz = UD_zz
//   UD_rz = -dz c ((r-rb) P0 + 2 rb Dc)    UK_rz = UD_rz
//                                          UK_zr =  dz c ((rb-r) P0 + 2 r Dc)
// Coincident points (s- <= 1e-20 s+) give zero (reading A2).
// PairEval is the same computation cut into stages (geometry -> Horner steps of the table -> finish) for kernels that
// interleave it with their DMMA stream; landau_tensor_2v runs the stages back to back.
// ------------------------------------------------------------------------------------------------------------
struct Tensor5 {
  double UDrr, UDrz, UDzz, UKrr, UKzr;
};

struct PairEval {
  double r, rb, dr, dz, rr4, ratio, c, m, x;
  EllipTable el;
  __device__ __forceinline__ void geometry(double r_, double z, double rb_, double zb, const double* __restrict__ tab) {
    r = r_;
    rb = rb_;
    dr = r - rb;
    dz = z - zb;
    double sm = fma(dr, dr, dz * dz);
    rr4 = 4.0 * r * rb;
    const double sp = sm + rr4;
    const bool coincident = sm <= 1e-20 * sp;
    sm = coincident ? sp : sm;
    const double inv = 1.0 / (sp * sm);
    const double isp = inv * sm;  // 1/s+
    x = sm * isp;                 // m' = s-/s+
    m = rr4 * isp;
    ratio = sp * sp * inv;        // s+/s-
    c = coincident ? 0.0 : 4.0 * isp * rsqrt(sp);
    el.start(x, tab);
  }
  template <int HI, int LO>
  __device__ __forceinline__ void steps() {
    el.template steps<HI, LO>();
  }
  __device__ __forceinline__ Tensor5 finish() {
    double E = el.E, Dc = el.Dc, Q = el.Q;
    if (x < ELLIP_TAB_XMIN) ellip_pieces_log(x, E, Dc, Q);  // near-coincident pairs only
    const double P0 = E * ratio;  // P0 = E / m'
    const double mP2 = m * (P0 - Dc - Q);
    const double dz2 = dz * dz;
    Tensor5 u;
    u.UDrr = c * fma(4.0 * rb * rb, Q, dz2 * P0);
    u.UDzz = c * fma(dr * dr, P0, rr4 * Dc);
    u.UDrz = -dz * c * fma(dr, P0, 2.0 * rb * Dc);
    u.UKrr = c * fma(rr4, Q, dz2 * mP2);
    u.UKzr = dz * c * fma(-dr, P0, 2.0 * r * Dc);
    return u;
  }
};

__device__ __forceinline__ Tensor5 landau_tensor_2v(double r, double z, double rb, double zb,
                                                    const double* __restrict__ tab = g_ellip_tab) {
  PairEval p;
  p.geometry(r, z, rb, zb, tab);
  p.template steps<LANDAU_ELLIP_TAB_DEG - 1, 0>();
  return p.finish();
}

__global__ void k_tensor_eval(const double* __restrict__ r, const double* __restrict__ z, const double* __restrict__ rb,
                              const double* __restrict__ zb, int n, double* __restrict__ out) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  Tensor5 u = landau_tensor_2v(r[t], z[t], rb[t], zb[t]);
  out[5 * t + 0] = u.UDrr;
  out[5 * t + 1] = u.UDrz;
  out[5 * t + 2] = u.UDzz;
  out[5 * t + 3] = u.UKrr;
  out[5 * t + 4] = u.UKzr;
}

__global__ void k_ellip_eval(const double* __restrict__ m, const double* __restrict__ mp, int n, double* __restrict__ out) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  double P0, Dc, Q;
  ellip_pieces(mp[t], P0, Dc, Q);
  P0 /= mp[t];
  out[3 * t + 0] = P0;
  out[3 * t + 1] = Dc;
  out[3 * t + 2] = Q;
}

// ------------------------------------------------------------------------------------------------------------
// Device-side description of one grid (pointers into context-owned tables).
// ------------------------------------------------------------------------------------------------------------
struct DevGrid {
  int n_cells, n_dof, n_ip, nnz;
  int ip_off;  // offset of this grid's IPs in the concatenated IP arrays
  const double* cell_sr;  // 2/hr per cell
  const double* cell_sz;  // 2/hz per cell
  const double* ip_w;     // [n_ip]
  const double* ip_gm;    // unstructured meshes: J^-T per point, [n_ip][4]; nullptr on rectangular grids (cell_sr / cell_sz)
  const int* en_ptr;      // [n_cells*nb + 1]
  const int* en_dof;
  const double* en_w;
  const int* as_ptr;  // [nnz+1]
  const int* as_code;
  const double* as_w;
  const int* ap_ptr;  // [n_dof+1]
  const int* ap_code;
  const double* ap_w;
};

// basis tabulation, [q][a]; nb, nq <= 25 (Q4)
struct DevTables {
  double B[640], dBxi[640], dBeta[640];
};

// ------------------------------------------------------------------------------------------------------------
// K1: source fields (kernel k1_fields below).
//   F layout: [col][3][nj_pad], col = col0 + b*ncb + c;  comp 0: w f, 1: w df/dr, 2: w df/dz
//   column c of the grid sums the species listed in (mix_ptr, mix_species, mix_wD, mix_wK).
// ------------------------------------------------------------------------------------------------------------
struct MixTable {  // per grid
  int ncb;         // columns per batch entry
  int n_entries;   // total entries
  int ptr[17];     // per column c: entries ptr[c]..ptr[c+1]   (ncb <= 16)
  int species_foff[16];  // offset of the species' dofs inside a batch entry
  double wD[16], wK[16];
};

constexpr int K2G_TJ = 16;

// offset (in doubles) of source value (col, comp, j) in the tiled F layout of a group with njt source tiles
__host__ __device__ __forceinline__ long long k2g_f_offset(int TC, int njt, int col, int comp, int j) {
  const int ct = col / TC, cl = col - ct * TC;
  const int jt = j >> 4, jj = j & 15;
  const int pos = (((jj >> 2) ^ (cl & 3)) << 2) | (jj & 3);
  return ((((long long)ct * njt + jt) * 3 + comp) * TC + cl) * 16 + pos;
}

// ------------------------------------------------------------------------------------------------------------
// K1: one CTA = one cell x 16 batch entries.  The cell's nodal values (constraints and species mix applied:
// fD = sum_e wD_e f_e for the value, fK = sum_e wK_e f_e for the gradient) are staged in shared memory once, then
// thread (q, entry) contracts them with the basis tabulation (stored [a][q]: conflict-free) and writes its three
// source values; the 16 points of a cell are contiguous in either F layout, so every warp store covers whole
// 128-byte lines.
// ------------------------------------------------------------------------------------------------------------
constexpr int K1T_BT = 16;

// NB basis functions, NQ integration points per cell (equal on tensor cells; 10 / 12 and 15 / 16 on P3 / P4 triangles)
template <int NB, int NQ = NB>
__global__ void __launch_bounds__(256)
k1_fields(DevGrid g, const DevTables* __restrict__ tab, MixTable mix, const double* __restrict__ batch_f,
               long long f_stride, int b0, int nbatch, double* __restrict__ F, long long nj_pad, int j_off_in_group,
               int col0, int tiled_tc) {
  constexpr int NQP = (NQ + 15) / 16 * 16;
  __shared__ double sT[3][NB][NQP];      // B, dBxi, dBeta as [a][q]
  __shared__ double sD[NB][K1T_BT], sK[NB][K1T_BT];
  const int tid = threadIdx.x, lo = tid & 15, bl = tid >> 4;
  const int cell = blockIdx.x, b = blockIdx.y * K1T_BT + bl;
  for (int e = tid; e < NQ * NB; e += 256) {
    const int q = e / NB, a = e - q * NB;
    sT[0][a][q] = tab->B[e];
    sT[1][a][q] = tab->dBxi[e];
    sT[2][a][q] = tab->dBeta[e];
  }
  const double sr = g.cell_sr[cell], sz = g.cell_sz[cell];
  const bool live = b < nbatch;
  const double* fb = batch_f + (long long)(b0 + (live ? b : 0)) * f_stride;
  for (int c = 0; c < mix.ncb; ++c) {
    __syncthreads();
    for (int a = lo; a < NB; a += 16) {  // basis function a (more than 16 on Q4: several per thread)
      double fD = 0.0, fK = 0.0;
      const int p0 = g.en_ptr[cell * NB + a], p1 = g.en_ptr[cell * NB + a + 1];
      for (int e = mix.ptr[c]; e < mix.ptr[c + 1]; ++e) {
        const double* fs = fb + mix.species_foff[e];
        double fa = 0.0;
        for (int p = p0; p < p1; ++p) fa = fma(g.en_w[p], fs[g.en_dof[p]], fa);
        fD = fma(mix.wD[e], fa, fD);
        fK = fma(mix.wK[e], fa, fK);
      }
      sD[a][bl] = fD;
      sK[a][bl] = fK;
    }
    __syncthreads();
    for (int q = lo; q < NQ && live; q += 16) {  // quadrature point q
      const int j = cell * NQ + q;
      const double w = g.ip_w[j];
      double v = 0.0, vx = 0.0, vy = 0.0;
#pragma unroll
      for (int a = 0; a < NB; ++a) {
        const double fd = sD[a][bl], fk = sK[a][bl];
        v = fma(sT[0][a][q], fd, v);
        vx = fma(sT[1][a][q], fk, vx);
        vy = fma(sT[2][a][q], fk, vy);
      }
      const long long col = col0 + (long long)b * mix.ncb + c;
      double gr = vx * sr, gz = vy * sz;
      if (g.ip_gm) {  // non-affine cell: (d/dr, d/dz) = J^-T (d/dxi, d/deta) at this point
        const double* m = g.ip_gm + 4 * (long long)j;
        gr = fma(m[0], vx, m[1] * vy);
        gz = fma(m[2], vx, m[3] * vy);
      }
      const double o0 = w * v, o1 = w * gr, o2 = w * gz;
      if (tiled_tc) {
        const int njt = (int)(nj_pad >> 4), jg = j_off_in_group + j;
        F[k2g_f_offset(tiled_tc, njt, (int)col, 0, jg)] = o0;
        F[k2g_f_offset(tiled_tc, njt, (int)col, 1, jg)] = o1;
        F[k2g_f_offset(tiled_tc, njt, (int)col, 2, jg)] = o2;
      } else {
        double* dst = F + col * 3 * nj_pad + j_off_in_group + j;
        dst[0] = o0;
        dst[nj_pad] = o1;
        dst[2 * nj_pad] = o2;
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------------------
// K2 (plain FP64 FMA): thread = one field point i, NC columns; the block's 128 field points share source tiles
// staged in shared memory (every lane reads the same address: broadcast).  blockIdx.z splits the j range.
//   G layout: [split][col][5][n_i]   comp: 0 GD_rr, 1 GD_rz, 2 GD_zz, 3 GK_r, 4 GK_z
// ------------------------------------------------------------------------------------------------------------
constexpr int K2_TJ = 16;  // source points per shared-memory tile

template <int NC>
__global__ void __launch_bounds__(128)
k2_inner_dfma(const double* __restrict__ ip_r, const double* __restrict__ ip_z, int n_i, int j0, int nj_pad,
              const double* __restrict__ F, int ncols, double* __restrict__ G, long long g_split_stride, int gcol0) {
  __shared__ double s_r[K2_TJ], s_z[K2_TJ];
  __shared__ double s_F[NC][3][K2_TJ];
  const int i = min((int)(blockIdx.x * blockDim.x + threadIdx.x), n_i - 1);
  const double r = ip_r[i], z = ip_z[i];
  const int colbase = blockIdx.y * NC;
  const int ntiles = nj_pad / K2_TJ;
  const int per = (ntiles + gridDim.z - 1) / gridDim.z;
  const int t0 = blockIdx.z * per, t1 = min(t0 + per, ntiles);
  double acc[NC][5];
#pragma unroll
  for (int c = 0; c < NC; ++c)
#pragma unroll
    for (int k = 0; k < 5; ++k) acc[c][k] = 0.0;
  for (int t = t0; t < t1; ++t) {
    __syncthreads();
    if (threadIdx.x < K2_TJ) {
      s_r[threadIdx.x] = ip_r[j0 + t * K2_TJ + threadIdx.x];
      s_z[threadIdx.x] = ip_z[j0 + t * K2_TJ + threadIdx.x];
    }
    for (int e = threadIdx.x; e < NC * 3 * K2_TJ; e += blockDim.x) {
      const int jj = e % K2_TJ, ck = e / K2_TJ;  // ck = c*3 + comp
      const int col = colbase + ck / 3;
      (&s_F[0][0][0])[e] = col < ncols ? F[((long long)col * 3 + ck % 3) * nj_pad + t * K2_TJ + jj] : 0.0;
    }
    __syncthreads();
#pragma unroll 2
    for (int jj = 0; jj < K2_TJ; ++jj) {
      const Tensor5 u = landau_tensor_2v(r, z, s_r[jj], s_z[jj]);
#pragma unroll
      for (int c = 0; c < NC; ++c) {
        const double wf = s_F[c][0][jj], wfr = s_F[c][1][jj], wfz = s_F[c][2][jj];
        acc[c][0] = fma(u.UDrr, wf, acc[c][0]);
        acc[c][1] = fma(u.UDrz, wf, acc[c][1]);
        acc[c][2] = fma(u.UDzz, wf, acc[c][2]);
        acc[c][3] = fma(u.UKrr, wfr, fma(u.UDrz, wfz, acc[c][3]));
        acc[c][4] = fma(u.UKzr, wfr, fma(u.UDzz, wfz, acc[c][4]));
      }
    }
  }
  if (blockIdx.x * blockDim.x + threadIdx.x < n_i) {
#pragma unroll
    for (int c = 0; c < NC; ++c)
      if (colbase + c < ncols) {
        double* dst = G + blockIdx.z * g_split_stride + ((long long)(gcol0 + colbase + c) * 5) * n_i + i;
#pragma unroll
        for (int k = 0; k < 5; ++k) dst[(long long)k * n_i] = acc[c][k];
      }
  }
}

// ------------------------------------------------------------------------------------------------------------
// K2 (DMMA): the inner integral as a GEMM whose A operand is generated on the fly.
//   G[i, comp, col] = sum_j U_comp(i,j) F[j, col]  -- per warp an 8(i) x 8NT(col) output tile, k = 4 source points per
//   step.  Lane (g = lane/4, t = lane%4) evaluates the tensor of the pair (i0+g, j+t): exactly the A-fragment
//   layout of mma.m8n8k4.f64, so the five tensor components go from registers straight into seven DMMAs per
//   8-column tile (3 for G^D, 4 for G^K) with no shared-memory round trip.  B fragments (F[j+t][col0+g]) come
//   from a shared-memory tile [col][3][TJ+4] (row stride 20 doubles: conflict-free), double-buffered with cp.async.
//   Block = 8 warps = 64 field points; blockIdx.y = column tile; blockIdx.z = j split.
// ------------------------------------------------------------------------------------------------------------
constexpr int K2M_TJ = 16;
constexpr int K2M_LD = K2M_TJ + 4;

__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N));
}

template <int NT>
__global__ void __launch_bounds__(256)
k2_inner_dmma(const double* __restrict__ ip_r, const double* __restrict__ ip_z, int n_i, int j0, int nj_pad,
              const double* __restrict__ F, int ncols_pad, int ncols, double* __restrict__ G, long long g_split_stride,
              int gcol0) {
  constexpr int CT = 8 * NT;
  extern __shared__ __align__(16) double smem[];
  // per stage: s_F[CT][3][K2M_LD], s_r[K2M_TJ], s_z[K2M_TJ]
  constexpr int STAGE = CT * 3 * K2M_LD + 2 * K2M_TJ;
  constexpr int TAB = 4 * LANDAU_ELLIP_TAB_BINADES * (LANDAU_ELLIP_TAB_DEG + 1) * 4;
  double* sTab = smem + 2 * STAGE;  // elliptic table T, copied once (visible after the first barrier of the tile loop)
  for (int e = threadIdx.x; e < TAB; e += 256) sTab[e] = g_ellip_tab[e];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int gq = lane >> 2, tq = lane & 3;
  const int i = min((int)(blockIdx.x * 64 + warp * 8 + gq), n_i - 1);
  const double r = ip_r[i], z = ip_z[i];
  const int colbase = blockIdx.y * CT;
  const int ntiles = nj_pad / K2M_TJ;
  const int per = (ntiles + gridDim.z - 1) / gridDim.z;
  const int t0 = blockIdx.z * per, t1 = min(t0 + per, ntiles);

  double acc[NT][5][2];
#pragma unroll
  for (int n = 0; n < NT; ++n)
#pragma unroll
    for (int k = 0; k < 5; ++k) acc[n][k][0] = acc[n][k][1] = 0.0;

  auto issue_tile = [&](int t, int stage) {
    double* sF = smem + stage * STAGE;
    // CT*3 rows of K2M_TJ doubles = 8 x 16-byte chunks per row
    for (int e = threadIdx.x; e < CT * 3 * (K2M_TJ / 2); e += 256) {
      const int row = e / (K2M_TJ / 2), ch = e % (K2M_TJ / 2);
      const double* src = F + ((long long)(colbase * 3 + row)) * nj_pad + (long long)t * K2M_TJ + ch * 2;
      cp_async16(sF + row * K2M_LD + ch * 2, src);
    }
    if (threadIdx.x < K2M_TJ / 2) {
      cp_async16(sF + CT * 3 * K2M_LD + threadIdx.x * 2, ip_r + j0 + t * K2M_TJ + threadIdx.x * 2);
    } else if (threadIdx.x < K2M_TJ) {
      const int c = threadIdx.x - K2M_TJ / 2;
      cp_async16(sF + CT * 3 * K2M_LD + K2M_TJ + c * 2, ip_z + j0 + t * K2M_TJ + c * 2);
    }
    cp_async_commit();
  };

  Tensor5 u = {0.0, 0.0, 0.0, 0.0, 0.0};
  if (t0 < t1) issue_tile(t0, 0);
  for (int t = t0; t < t1; ++t) {
    const int stage = (t - t0) & 1;
    if (t + 1 < t1) {
      issue_tile(t + 1, stage ^ 1);
      cp_async_wait<1>();
    } else {
      cp_async_wait<0>();
    }
    __syncthreads();
    const double* sF = smem + stage * STAGE;
    const double* s_r = sF + CT * 3 * K2M_LD;
    const double* s_z = s_r + K2M_TJ;
    // the tensor of the NEXT four source points is evaluated in stages between the DMMAs of the current four
    // (PairEval: geometry, three Horner thirds, finish), so that its dependent FP64 chain hides under the DMMA stream;
    // across a tile boundary the next points' coordinates come from global memory, fetched a whole tile earlier;
    // only the very first four points are evaluated up front
    constexpr int D = LANDAU_ELLIP_TAB_DEG, H1 = D - 1 - D / 3, H2 = H1 - D / 3;
    if (t == t0) u = landau_tensor_2v(r, z, s_r[tq], s_z[tq], sTab);
    const bool next_tile = t + 1 < t1;
    const double rn = next_tile ? ip_r[j0 + (t + 1) * K2M_TJ + tq] : 1.0, zn = next_tile ? ip_z[j0 + (t + 1) * K2M_TJ + tq] : 0.0;
#pragma unroll
    for (int jj = 0; jj < K2M_TJ; jj += 4) {
      const bool inner = jj + 4 < K2M_TJ;
      const bool more = inner || next_tile;
      PairEval pe;
      if (more) pe.geometry(r, z, inner ? s_r[(jj + 4) % K2M_TJ + tq] : rn, inner ? s_z[(jj + 4) % K2M_TJ + tq] : zn, sTab);
#pragma unroll
      for (int n = 0; n < NT; ++n) {
        const double* col = sF + ((n * 8 + gq) * 3) * K2M_LD + jj + tq;
        const double wf = col[0], wfr = col[K2M_LD], wfz = col[2 * K2M_LD];
        dmma884(acc[n][0][0], acc[n][0][1], u.UDrr, wf);
        dmma884(acc[n][1][0], acc[n][1][1], u.UDrz, wf);
        dmma884(acc[n][2][0], acc[n][2][1], u.UDzz, wf);
        dmma884(acc[n][3][0], acc[n][3][1], u.UKrr, wfr);
        dmma884(acc[n][3][0], acc[n][3][1], u.UDrz, wfz);
        dmma884(acc[n][4][0], acc[n][4][1], u.UKzr, wfr);
        dmma884(acc[n][4][0], acc[n][4][1], u.UDzz, wfz);
        if (more) {
          if (n == (NT - 1) / 4) pe.template steps<D - 1, H1 + 1>();
          if (n == (NT - 1) / 2) pe.template steps<H1, H2 + 1>();
          if (n == (3 * (NT - 1)) / 4) pe.template steps<H2, 0>();
        }
      }
      if (more) u = pe.finish();
    }
    __syncthreads();
  }
  // C fragment: row gq (field point), columns 2 tq, 2 tq + 1
  if (blockIdx.x * 64 + warp * 8 + gq < n_i) {
#pragma unroll
    for (int n = 0; n < NT; ++n)
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int col = colbase + n * 8 + 2 * tq + h;
        if (col < ncols) {
          double* dst = G + blockIdx.z * g_split_stride + ((long long)(gcol0 + col) * 5) * n_i + i;
#pragma unroll
          for (int k = 0; k < 5; ++k) dst[(long long)k * n_i] = acc[n][k][h];
        }
      }
  }
}

}  // namespace landau
#include "k2_gemm.cuh"
namespace landau {

// ------------------------------------------------------------------------------------------------------------
// K2b: species combination (eq. 2.1 prefactors) and sum over j splits.
//   DK[b][species a][5][n_ip(g(a))] = sum_terms coef * sum_split G[split][col][comp][ip_off + i]
// ------------------------------------------------------------------------------------------------------------
struct CombineTable {   // per species alpha
  int n_terms;
  int col_base[16];     // column of batch entry 0
  int col_stride[16];   // columns per batch entry of that group
  double coefD[16], coefK[16];
  int ip_off, n_ip;     // the species' grid: offset in the concatenated IP arrays, number of IPs
  long long dk_off;     // offset of the species' block inside one entry of DK
  const double* ip_gm;  // the grid's J^-T per point (unstructured meshes) or nullptr
};

// one launch for all species: blockIdx.z = species
__global__ void __launch_bounds__(256)
k2b_combine(const CombineTable* __restrict__ cts, const double* __restrict__ G, long long g_split_stride, int n_split,
            int n_i_total, int nbatch, double* __restrict__ DK, long long dk_stride) {
  const CombineTable& ct = cts[blockIdx.z];
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int b = blockIdx.y;
  const int ip_off = ct.ip_off, n_ip = ct.n_ip;
  const long long dk_off = ct.dk_off;
  if (i >= n_ip || b >= nbatch) return;
  double out[5] = {0, 0, 0, 0, 0};
  for (int t = 0; t < ct.n_terms; ++t) {
    const long long col = ct.col_base[t] + (long long)b * ct.col_stride[t];
    double s[5] = {0, 0, 0, 0, 0};
    for (int sp = 0; sp < n_split; ++sp) {
      const double* src = G + sp * g_split_stride + col * 5 * n_i_total + ip_off + i;
#pragma unroll
      for (int k = 0; k < 5; ++k) s[k] += src[(long long)k * n_i_total];
    }
    out[0] = fma(ct.coefD[t], s[0], out[0]);
    out[1] = fma(ct.coefD[t], s[1], out[1]);
    out[2] = fma(ct.coefD[t], s[2], out[2]);
    out[3] = fma(ct.coefK[t], s[3], out[3]);
    out[4] = fma(ct.coefK[t], s[4], out[4]);
  }
  if (ct.ip_gm) {
    // unstructured mesh: K3 and K3' work in reference coordinates there, so D and K are pulled back,
    // D~ = M^T D M, K~ = M^T K with M = J^-T of this point (grad phi = M grad_ref phi)
    const double* m = ct.ip_gm + 4 * (long long)i;
    const double m00 = m[0], m01 = m[1], m10 = m[2], m11 = m[3];
    const double drr = out[0], drz = out[1], dzz = out[2], kr = out[3], kz = out[4];
    out[0] = m00 * (m00 * drr + m10 * drz) + m10 * (m00 * drz + m10 * dzz);
    out[1] = m01 * (m00 * drr + m10 * drz) + m11 * (m00 * drz + m10 * dzz);
    out[2] = m01 * (m01 * drr + m11 * drz) + m11 * (m01 * drz + m11 * dzz);
    out[3] = m00 * kr + m10 * kz;
    out[4] = m01 * kr + m11 * kz;
  }
  double* dst = DK + (long long)b * dk_stride + dk_off + i;
#pragma unroll
  for (int k = 0; k < 5; ++k) dst[(long long)k * n_ip] = out[k];
}

// ------------------------------------------------------------------------------------------------------------
// K3: one thread per CSR slot of (batch entry, species): gathers its element-matrix contributions, each formed
// on the fly  A_e[a][c] = sum_q w_q [ phi_a phi_c / dt + grad phi_a . D grad phi_c - (grad phi_a . K) phi_c ]
// (eq. 2.4 with the sparse Jacobian of PAPER.md:73), weighted by the constraint products P[a][I] P[c][J].
// Every CSR value is written exactly once, coalesced along the slot index; no atomics.
// ------------------------------------------------------------------------------------------------------------
template <int NB, int NQ = NB>
__global__ void __launch_bounds__(256)
k3_assemble(DevGrid g, const DevTables* __restrict__ tab, const double* __restrict__ DK, long long dk_stride,
            long long dk_off, double inv_dt, int nbatch, double* __restrict__ vals, long long v_stride, long long v_off) {
  __shared__ double sB[NQ * NB], sX[NQ * NB], sY[NQ * NB];
  for (int e = threadIdx.x; e < NQ * NB; e += blockDim.x) {
    sB[e] = tab->B[e];
    sX[e] = tab->dBxi[e];
    sY[e] = tab->dBeta[e];
  }
  __syncthreads();
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  const int b = blockIdx.y;
  if (n >= g.nnz || b >= nbatch) return;
  const double* dk = DK + (long long)b * dk_stride + dk_off;
  double total = 0.0;
  for (int p = g.as_ptr[n]; p < g.as_ptr[n + 1]; ++p) {
    const int code = g.as_code[p];
    const int c = code % NB, a = (code / NB) % NB, cell = code / (NB * NB);
    const double sr = g.cell_sr[cell], sz = g.cell_sz[cell];
    double s = 0.0;
#pragma unroll 4
    for (int q = 0; q < NQ; ++q) {
      const int ip = cell * NQ + q;
      const double w = g.ip_w[ip];
      const double Drr = dk[ip], Drz = dk[g.n_ip + ip], Dzz = dk[2 * g.n_ip + ip], Kr = dk[3 * g.n_ip + ip],
                   Kz = dk[4 * g.n_ip + ip];
      const double pa = sB[q * NB + a], par = sX[q * NB + a] * sr, paz = sY[q * NB + a] * sz;
      const double pc = sB[q * NB + c], pcr = sX[q * NB + c] * sr, pcz = sY[q * NB + c] * sz;
      double v = inv_dt * pa * pc;
      v = fma(par, fma(Drr, pcr, Drz * pcz), v);
      v = fma(paz, fma(Drz, pcr, Dzz * pcz), v);
      v = fma(-fma(par, Kr, paz * Kz), pc, v);
      s = fma(w, v, s);
    }
    total = fma(g.as_w[p], s, total);
  }
  vals[(long long)b * v_stride + v_off + n] = total;
}

// ------------------------------------------------------------------------------------------------------------
// K3 for cells without a ring schedule (triangles, grids the ring does not fit): element matrices first, then a gather.
//   k3_elem_matrix: one CTA = one cell x K3E_BT batch entries of one species; thread (a, c) forms the six products of its
//     two basis functions per point once and applies them to the (w D, w K) of every entry (staged in shared memory, read
//     as broadcasts):  A_e[a][c] = sum_q w_q [ phi_a phi_c / dt + grad phi_a . D grad phi_c - (grad phi_a . K) phi_c ]
//     -> scratch EM[entry][species][cell][NB x NB]   (each D, K value is used NB^2 times instead of being re-read per slot).
//   k3_gather: one thread per CSR slot and K3G_BT entries sums the slot's (constraint weight, matrix entry) list -- the codes
//     of the slot lists, (cell NB + a) NB + c, are the offsets into a species' scratch block.  Written once, no atomics.
// ------------------------------------------------------------------------------------------------------------
constexpr int K3E_BT = 8, K3G_BT = 8;

template <int NB, int NQ = NB>
__global__ void __launch_bounds__(256)
k3_elem_matrix(DevGrid g, const DevTables* __restrict__ tab, const double* __restrict__ DK, long long dk_stride,
               long long dk_off, double inv_dt, int nbatch, double* __restrict__ EM, long long em_stride, long long em_off) {
  __shared__ double sB[NQ * NB], sX[NQ * NB], sY[NQ * NB];
  __shared__ double sDK[K3E_BT][NQ][5];  // w Drr, w Drz, w Dzz, w Kr, w Kz
  __shared__ double sW[NQ];
  const int tid = threadIdx.x, cell = blockIdx.x, b0 = blockIdx.y * K3E_BT;
  const double sr = g.cell_sr[cell], sz = g.cell_sz[cell];
  for (int e = tid; e < NQ * NB; e += 256) {
    sB[e] = tab->B[e];
    sX[e] = tab->dBxi[e] * sr;
    sY[e] = tab->dBeta[e] * sz;
  }
  if (tid < NQ) sW[tid] = g.ip_w[cell * NQ + tid];
  for (int e = tid; e < K3E_BT * NQ * 5; e += 256) {
    const int k = e % 5, q = (e / 5) % NQ, bl = e / (5 * NQ);
    const int ip = cell * NQ + q;
    sDK[bl][q][k] = b0 + bl < nbatch ? g.ip_w[ip] * DK[(long long)(b0 + bl) * dk_stride + dk_off + (long long)k * g.n_ip + ip] : 0.0;
  }
  __syncthreads();
  for (int e = tid; e < NB * NB; e += 256) {  // one (a, c) per thread up to Q3 / P4, three on Q4
    const int a = e / NB, c = e - a * NB;
    double acc[K3E_BT], mass = 0.0;
#pragma unroll
    for (int bl = 0; bl < K3E_BT; ++bl) acc[bl] = 0.0;
#pragma unroll 2
    for (int q = 0; q < NQ; ++q) {
      const double pa = sB[q * NB + a], par = sX[q * NB + a], paz = sY[q * NB + a];
      const double pc = sB[q * NB + c], pcr = sX[q * NB + c], pcz = sY[q * NB + c];
      const double m_rr = par * pcr, m_rz = fma(par, pcz, paz * pcr), m_zz = paz * pcz, m_r = -par * pc, m_z = -paz * pc;
      mass = fma(sW[q], pa * pc, mass);
#pragma unroll
      for (int bl = 0; bl < K3E_BT; ++bl) {
        const double* d = sDK[bl][q];
        acc[bl] = fma(d[0], m_rr, fma(d[1], m_rz, fma(d[2], m_zz, fma(d[3], m_r, fma(d[4], m_z, acc[bl])))));
      }
    }
    double* dst = EM + (long long)b0 * em_stride + em_off + (long long)cell * (NB * NB) + e;
#pragma unroll
    for (int bl = 0; bl < K3E_BT; ++bl)
      if (b0 + bl < nbatch) dst[bl * em_stride] = fma(inv_dt, mass, acc[bl]);
  }
}

// grid (ceil(nnz / 256), ceil(nbatch / K3G_BT)) per species
__global__ void __launch_bounds__(256)
k3_gather(DevGrid g, int nbatch, const double* __restrict__ EM, long long em_stride, long long em_off,
          double* __restrict__ vals, long long v_stride, long long v_off) {
  const int n = blockIdx.x * 256 + threadIdx.x, b0 = blockIdx.y * K3G_BT;
  if (n >= g.nnz) return;
  const double* em = EM + (long long)b0 * em_stride + em_off;
  double v[K3G_BT];
#pragma unroll
  for (int k = 0; k < K3G_BT; ++k) v[k] = 0.0;
  const int p1 = g.as_ptr[n + 1], nb = min(K3G_BT, nbatch - b0);
  for (int p = g.as_ptr[n]; p < p1; ++p) {
    const double w = g.as_w[p];
    const double* src = em + g.as_code[p];
#pragma unroll
    for (int k = 0; k < K3G_BT; ++k)
      if (k < nb) v[k] = fma(w, src[k * em_stride], v[k]);
  }
  double* dst = vals + (long long)b0 * v_stride + v_off + n;
#pragma unroll
  for (int k = 0; k < K3G_BT; ++k)
    if (k < nb) __stcs(dst + k * v_stride, v[k]);
}

// ------------------------------------------------------------------------------------------------------------
// K3' (apply):  rhs_a = - sum_q w_q grad phi_a . (D grad f - K f).
//   k3_elem_apply: one CTA = one cell x 16 batch entries (as K1): nodal values staged in shared memory, thread
//     (q, entry) forms f, grad f and the weighted flux at its point, thread (a, entry) contracts the fluxes with the
//     basis gradients -> element vector RE[entry][cell * NB + a] (contiguous 128-byte lines per entry).
//   k3_apply_gather: one thread per (dof, entry) sums its element-vector entries (constraint weights), coalesced along
//     the dof index.
// ------------------------------------------------------------------------------------------------------------
// One launch for all species of a context (a Newton iteration applies the operator to every species: ten launch pairs on
// the paper's ten-species problem became one pair): thread blocks are dealt to species by prefix sums of their cell /
// dof-block counts.
struct ApplySpecies {
  DevGrid g;
  long long f_off, dk_off, re_off;
  int cell_end;    // exclusive prefix sum of n_cells over the species up to and including this one
  int dofblk_end;  // the same for ceil(n_dof / 256)
};

template <int NB, int NQ>
__device__ __forceinline__ void k3_elem_apply_body(const DevGrid& g, const DevTables* __restrict__ tab,
                                                   const double* __restrict__ batch_f, long long f_stride, long long f_off, int b0,
                                                   const double* __restrict__ DK, long long dk_stride, long long dk_off, int nbatch,
                                                   double* __restrict__ RE, long long re_stride, long long re_off, int cell) {
  constexpr int NQP = (NQ + 15) / 16 * 16;
  __shared__ double sT[3][NB][NQP];  // B, dBxi, dBeta as [a][q]
  __shared__ double sF[NB][K1T_BT], sFl[2][NQ][K1T_BT];
  const int tid = threadIdx.x, lo = tid & 15, bl = tid >> 4;
  const int b = blockIdx.y * K1T_BT + bl;
  const bool live = b < nbatch;
  for (int e = tid; e < NQ * NB; e += 256) {
    const int q = e / NB, a = e - q * NB;
    sT[0][a][q] = tab->B[e];
    sT[1][a][q] = tab->dBxi[e];
    sT[2][a][q] = tab->dBeta[e];
  }
  const double sr = g.cell_sr[cell], sz = g.cell_sz[cell];
  for (int a = lo; a < NB; a += 16) {  // basis function a: constrained nodal value
    const double* fs = batch_f + (long long)(b0 + (live ? b : 0)) * f_stride + f_off;
    double fa = 0.0;
    for (int p = g.en_ptr[cell * NB + a]; p < g.en_ptr[cell * NB + a + 1]; ++p) fa = fma(g.en_w[p], fs[g.en_dof[p]], fa);
    sF[a][bl] = fa;
  }
  __syncthreads();
  for (int q = lo; q < NQ; q += 16) {  // quadrature point q
    double v = 0.0, vx = 0.0, vy = 0.0;
#pragma unroll
    for (int a = 0; a < NB; ++a) {
      const double fa = sF[a][bl];
      v = fma(sT[0][a][q], fa, v);
      vx = fma(sT[1][a][q], fa, vx);
      vy = fma(sT[2][a][q], fa, vy);
    }
    const int j = cell * NQ + q;
    const double fr = vx * sr, fz = vy * sz, w = g.ip_w[j];
    const double* dk = DK + (long long)(live ? b : 0) * dk_stride + dk_off;
    const double Drr = dk[j], Drz = dk[g.n_ip + j], Dzz = dk[2 * g.n_ip + j], Kr = dk[3 * g.n_ip + j], Kz = dk[4 * g.n_ip + j];
    sFl[0][q][bl] = w * (fma(Drr, fr, Drz * fz) - Kr * v);
    sFl[1][q][bl] = w * (fma(Drz, fr, Dzz * fz) - Kz * v);
  }
  __syncthreads();
  for (int a = lo; a < NB && live; a += 16) {  // basis function a again
    double r = 0.0;
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
      r = fma(sT[1][a][q] * sr, sFl[0][q][bl], r);
      r = fma(sT[2][a][q] * sz, sFl[1][q][bl], r);
    }
    RE[(long long)b * re_stride + re_off + cell * NB + a] = r;
  }
}

// blockIdx.x runs over the cells of all species
template <int NB, int NQ = NB>
__global__ void __launch_bounds__(256)
k3_elem_apply_all(const ApplySpecies* __restrict__ spec, int n_spec, const DevTables* __restrict__ tab,
                  const double* __restrict__ batch_f, long long f_stride, int b0, const double* __restrict__ DK,
                  long long dk_stride, int nbatch, double* __restrict__ RE, long long re_stride) {
  int s = 0;
  while (s + 1 < n_spec && (int)blockIdx.x >= spec[s].cell_end) ++s;
  const ApplySpecies& sp = spec[s];
  const int cell = blockIdx.x - (s ? spec[s - 1].cell_end : 0);
  k3_elem_apply_body<NB, NQ>(sp.g, tab, batch_f, f_stride, sp.f_off, b0, DK, dk_stride, sp.dk_off, nbatch, RE, re_stride, sp.re_off,
                             cell);
}

__device__ __forceinline__ void k3_apply_gather_body(const DevGrid& g, const double* __restrict__ RE, long long re_stride,
                                                     long long re_off, int nbatch, double* __restrict__ rhs, long long f_stride,
                                                     long long f_off, int b0, int n) {
  const int b = blockIdx.y;
  if (n >= g.n_dof || b >= nbatch) return;
  const double* re = RE + (long long)b * re_stride + re_off;
  double total = 0.0;
  for (int p = g.ap_ptr[n]; p < g.ap_ptr[n + 1]; ++p) total = fma(g.ap_w[p], re[g.ap_code[p]], total);
  rhs[(long long)(b0 + b) * f_stride + f_off + n] = -total;
}

// blockIdx.x runs over the 256-dof blocks of all species
__global__ void __launch_bounds__(256)
k3_apply_gather_all(const ApplySpecies* __restrict__ spec, int n_spec, const double* __restrict__ RE, long long re_stride,
                    int nbatch, double* __restrict__ rhs, long long f_stride, int b0) {
  int s = 0;
  while (s + 1 < n_spec && (int)blockIdx.x >= spec[s].dofblk_end) ++s;
  const ApplySpecies& sp = spec[s];
  const int blk = blockIdx.x - (s ? spec[s - 1].dofblk_end : 0);
  k3_apply_gather_body(sp.g, RE, re_stride, sp.re_off, nbatch, rhs, f_stride, sp.f_off, b0, blk * blockDim.x + threadIdx.x);
}

// ------------------------------------------------------------------------------------------------------------
// FP64 pipe probes (roofline denominators measured in-process by bench.py).
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_probe_dfma(double* out, int iters, double a, double b) {
  double acc[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) acc[k] = threadIdx.x * 1e-3 + k;
  for (int it = 0; it < iters; ++it)
#pragma unroll
    for (int u = 0; u < 8; ++u)
#pragma unroll
      for (int k = 0; k < 8; ++k) acc[k] = fma(acc[k], a, b);
  double s = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += acc[k];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void __launch_bounds__(256) k_probe_dmma(double* out, int iters, double a, double b) {
  double c0[8], c1[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    c0[k] = threadIdx.x * 1e-3 + k;
    c1[k] = k;
  }
  for (int it = 0; it < iters; ++it)
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
      for (int k = 0; k < 8; ++k) dmma884(c0[k], c1[k], a, b);
  double s = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += c0[k] + c1[k];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// mixed: 8 independent DFMA chains + 4 DMMA accumulator pairs per round -- are the two pipes concurrent?
// L2 -> SM read bandwidth (the roofline denominator of the solve on systems whose matrix values stream from L2): every
// thread block sweeps the whole buffer `iters` times with 16-byte loads that bypass L1 (ld.global.cg)
__global__ void __launch_bounds__(256) k_probe_l2_read(const double2* __restrict__ buf, long long n16, int iters, double* out) {
  double acc = 0.0;
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (int it = 0; it < iters; ++it) {
#pragma unroll 8
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n16; i += stride) {
      const double2 v = __ldcg(buf + i);
      acc += v.x + v.y;
    }
  }
  out[blockIdx.x * (long long)blockDim.x + threadIdx.x] = acc;
}

__global__ void __launch_bounds__(256) k_probe_mixed(double* out, int iters, double a, double b) {
  double acc[8], c0[4], c1[4];
#pragma unroll
  for (int k = 0; k < 8; ++k) acc[k] = threadIdx.x * 1e-3 + k;
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    c0[k] = threadIdx.x * 1e-3 + k;
    c1[k] = k;
  }
  for (int it = 0; it < iters; ++it)
#pragma unroll
    for (int u = 0; u < 4; ++u) {
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        dmma884(c0[k], c1[k], a, b);
        acc[2 * k] = fma(acc[2 * k], a, b);
        acc[2 * k + 1] = fma(acc[2 * k + 1], a, b);
      }
    }
  double s = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += acc[k];
#pragma unroll
  for (int k = 0; k < 4; ++k) s += c0[k] + c1[k];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace landau
