// landau3v_api.cu -- the C ABI of include/landau3v.h: context, scratch management and kernel launches of the 3V variant.
#include <cmath>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include <nvtx3/nvToolsExt.h>

#include "../../include/landau3v.h"
#include "batch_solver.hpp"
#include "host_setup3v.hpp"
#include "landau3v_kernels.cuh"
#include "landau3v_dmma.cuh"
#include "landau3v_k3.cuh"

using namespace landau3v;

namespace {
std::string g_create_error3;
}

struct landau3v_ctx {
  int device = 0, S = 0, G = 0, n_sm = 148;
  HostTables3 ht;
  std::vector<HostGrid3> hg;
  std::vector<landau_species_desc> species;
  std::vector<double> nu;
  bool separable = false;
  int n_classes = 1;  // source column classes: 1 (rank-one nu) or S
  std::vector<long long> f_off, v_off, dk_off, fe_off;
  long long f_stride = 0, v_stride = 0, dk_stride = 0, fe_stride = 0;
  std::vector<int> ip_off;
  int n_ip_total = 0, n_pad = 0, max_ip = 0;
  std::vector<void*> allocs;
  Tables3* d_tab = nullptr;
  std::vector<DevGrid3> dg;
  std::vector<const int*> d_rowptr, d_colidx;
  double *d_px = nullptr, *d_py = nullptr, *d_pz = nullptr;
  std::vector<Mix3> mix;
  Ranges3 ranges;
  Combine3* d_comb = nullptr;
  DevGrid3* d_grids = nullptr;
  Spec3* d_spec = nullptr;
  int max_cells = 0, max_nnz = 0;
  double* EM = nullptr;
  size_t EM_cap = 0;
  std::vector<long long> em_off;
  long long em_stride = 0;
  int dmma_ctas_per_sm[5] = {0, 0, 0, 0, 0}, dmma_stream_ctas_per_sm[5] = {0, 0, 0, 0, 0};
  double* part_buf = nullptr;  // stream mode of the DMMA inner integral: accumulator parts of cut items + arrival counters
  size_t part_cap = 0;
  int assembly_kernel = 0;  // 0: element matrices on the MMA pipe + gather, 1: per-slot quadrature (first version)
  bool k3e_configured = false;
  int k3e_ctas_per_sm = 0;
  double *F = nullptr, *Gs = nullptr, *DK = nullptr, *FE = nullptr, *stage_in = nullptr, *stage_out = nullptr;
  size_t F_cap = 0, G_cap = 0, DK_cap = 0, FE_cap = 0, stage_in_cap = 0, stage_out_cap = 0;
  int f_nbc = -1;
  int chunk = 256, inner_kernel = 0, last_batch = 0;
  cudaStream_t last_stream = nullptr;
  bool timing = false;
  std::vector<cudaEvent_t> ev;
  int ev_used = 0;
  long long launches = 0;
  // batched solve and implicit step (batch_solver.hpp); mass values of one entry, computed at the first landau3v_step
  landau::BatchSolver solver;
  double* st_M = nullptr;
  size_t st_M_cap = 0;
  std::string err;
};

namespace {

int fail(landau3v_ctx* ctx, int code, const std::string& msg) {
  if (ctx)
    ctx->err = msg;
  else
    g_create_error3 = msg;
  return code;
}

#define CUDA_TRY3(ctx, expr)                                                                      \
  do {                                                                                            \
    cudaError_t e_ = (expr);                                                                      \
    if (e_ != cudaSuccess)                                                                        \
      return fail(ctx, e_ == cudaErrorMemoryAllocation ? LANDAU_OUT_OF_MEMORY : LANDAU_CUDA_ERROR, \
                  std::string(#expr) + ": " + cudaGetErrorString(e_));                            \
  } while (0)

template <class T>
int upload(landau3v_ctx* ctx, const std::vector<T>& h, const T** out) {
  T* d = nullptr;
  CUDA_TRY3(ctx, cudaMalloc(&d, sizeof(T) * (h.empty() ? 1 : h.size())));
  ctx->allocs.push_back(d);
  if (!h.empty()) CUDA_TRY3(ctx, cudaMemcpy(d, h.data(), sizeof(T) * h.size(), cudaMemcpyHostToDevice));
  *out = d;
  return LANDAU_OK;
}

int grow(landau3v_ctx* ctx, double** p, size_t* cap, size_t need) {
  if (need <= *cap) return LANDAU_OK;
  if (*p) {
    CUDA_TRY3(ctx, cudaDeviceSynchronize());
    CUDA_TRY3(ctx, cudaFree(*p));
    *p = nullptr;
    *cap = 0;
  }
  CUDA_TRY3(ctx, cudaMalloc(p, need * sizeof(double)));
  *cap = need;
  return LANDAU_OK;
}

void mark(landau3v_ctx* ctx, cudaStream_t st) {
  if (!ctx->timing) return;
  if (ctx->ev_used == (int)ctx->ev.size()) {
    cudaEvent_t e = nullptr;
    cudaEventCreate(&e);
    ctx->ev.push_back(e);
  }
  cudaEventRecord(ctx->ev[ctx->ev_used++], st);
}

bool rank_one(const std::vector<double>& nu, int S, std::vector<double>* a, std::vector<double>* b) {
  int pr = -1, pc = -1;
  for (int i = 0; i < S && pr < 0; ++i)
    for (int j = 0; j < S; ++j)
      if (nu[i * S + j] != 0.0) {
        pr = i;
        pc = j;
        break;
      }
  a->assign(S, 0.0);
  b->assign(S, 0.0);
  if (pr < 0) return true;
  for (int j = 0; j < S; ++j) (*b)[j] = nu[pr * S + j];
  for (int i = 0; i < S; ++i) (*a)[i] = nu[i * S + pc] / nu[pr * S + pc];
  for (int i = 0; i < S; ++i)
    for (int j = 0; j < S; ++j) {
      const double ref = (*a)[i] * (*b)[j];
      if (std::fabs(nu[i * S + j] - ref) > 1e-14 * std::fabs(ref) + 1e-300) return false;
    }
  return true;
}

int build_device_side(landau3v_ctx* ctx) {
  const int G = ctx->G, S = ctx->S;
  Tables3* ht = new Tables3();
  for (int e = 0; e < 729; ++e) {
    ht->B[e] = ctx->ht.B[e];
    ht->dBx[e] = ctx->ht.dBx[e];
    ht->dBy[e] = ctx->ht.dBy[e];
    ht->dBz[e] = ctx->ht.dBz[e];
  }
  cudaError_t e1 = cudaMalloc(&ctx->d_tab, sizeof(Tables3));
  if (e1 == cudaSuccess) {
    ctx->allocs.push_back(ctx->d_tab);
    e1 = cudaMemcpy(ctx->d_tab, ht, sizeof(Tables3), cudaMemcpyHostToDevice);
  }
  delete ht;
  CUDA_TRY3(ctx, e1);
  // concatenated integration points, padded to whole tiles; padding points sit far away and carry F = 0
  const int tile = 128;
  ctx->n_pad = (ctx->n_ip_total + tile - 1) / tile * tile;
  std::vector<double> x(ctx->n_pad, 1e3), y(ctx->n_pad, 1e3), z(ctx->n_pad, 1e3);
  for (int g = 0; g < G; ++g)
    for (int j = 0; j < ctx->hg[g].n_ip; ++j) {
      x[ctx->ip_off[g] + j] = ctx->hg[g].ip_x[j];
      y[ctx->ip_off[g] + j] = ctx->hg[g].ip_y[j];
      z[ctx->ip_off[g] + j] = ctx->hg[g].ip_z[j];
    }
  const double* tmp;
  if (int rc = upload(ctx, x, &tmp)) return rc;
  ctx->d_px = const_cast<double*>(tmp);
  if (int rc = upload(ctx, y, &tmp)) return rc;
  ctx->d_py = const_cast<double*>(tmp);
  if (int rc = upload(ctx, z, &tmp)) return rc;
  ctx->d_pz = const_cast<double*>(tmp);
  ctx->dg.resize(G);
  ctx->d_rowptr.resize(G);
  ctx->d_colidx.resize(G);
  for (int g = 0; g < G; ++g) {
    const HostGrid3& h = ctx->hg[g];
    DevGrid3& d = ctx->dg[g];
    d.n_cells = h.n_cells;
    d.n_dof = h.n_dof;
    d.n_ip = h.n_ip;
    d.nnz = h.nnz;
    d.ip_off = ctx->ip_off[g];
    int rc = 0;
    rc = rc ? rc : upload(ctx, h.cell_h, &d.cell_h);
    rc = rc ? rc : upload(ctx, h.ip_w, &d.ip_w);
    rc = rc ? rc : upload(ctx, h.en_ptr, &d.en_ptr);
    rc = rc ? rc : upload(ctx, h.en_dof, &d.en_dof);
    rc = rc ? rc : upload(ctx, h.en_w, &d.en_w);
    rc = rc ? rc : upload(ctx, h.as_ptr, &d.as_ptr);
    rc = rc ? rc : upload(ctx, h.as_code, &d.as_code);
    rc = rc ? rc : upload(ctx, h.as_w, &d.as_w);
    rc = rc ? rc : upload(ctx, h.ap_ptr, &d.ap_ptr);
    rc = rc ? rc : upload(ctx, h.ap_code, &d.ap_code);
    rc = rc ? rc : upload(ctx, h.ap_w, &d.ap_w);
    rc = rc ? rc : upload(ctx, h.rowptr, &ctx->d_rowptr[g]);
    rc = rc ? rc : upload(ctx, h.colidx, &ctx->d_colidx[g]);
    if (rc) return rc;
  }
  // source column classes, mixing weights, combination tables
  std::vector<double> sa, sb;
  ctx->separable = rank_one(ctx->nu, S, &sa, &sb);
  ctx->n_classes = ctx->separable ? 1 : S;
  ctx->mix.assign(G, Mix3());
  for (int g = 0; g < G; ++g) {
    Mix3& m = ctx->mix[g];
    memset(&m, 0, sizeof(m));
    for (int s = 0; s < S; ++s)
      if (ctx->species[s].grid == g) {
        if (m.n_entries >= MAX_TERMS) return fail(ctx, LANDAU_UNSUPPORTED, "more than 16 species on one grid");
        const int n = m.n_entries++;
        m.cls[n] = ctx->separable ? 0 : s;
        m.f_off[n] = (int)ctx->f_off[s];
        m.wD[n] = ctx->separable ? sb[s] : 1.0;
        m.wK[n] = (ctx->separable ? sb[s] : 1.0) / ctx->species[s].mass;
      }
  }
  memset(&ctx->ranges, 0, sizeof(ctx->ranges));
  for (int c = 0; c < ctx->n_classes; ++c) {
    const int g = ctx->species[c].grid;
    const int lo = ctx->separable ? 0 : ctx->ip_off[g], hi = ctx->separable ? ctx->n_ip_total : ctx->ip_off[g + 1];
    ctx->ranges.j0[c] = lo / K2_TJ * K2_TJ;
    ctx->ranges.j1[c] = std::min(ctx->n_pad, (hi + K2_TJ - 1) / K2_TJ * K2_TJ);
  }
  std::vector<Combine3> comb(S);
  for (int s = 0; s < S; ++s) {
    Combine3& c = comb[s];
    memset(&c, 0, sizeof(c));
    const int g = ctx->species[s].grid;
    const double ma = ctx->species[s].mass;
    c.ip_off = ctx->ip_off[g];
    c.n_ip = ctx->hg[g].n_ip;
    c.dk_off = ctx->dk_off[s];
    if (ctx->separable) {
      c.n_terms = 1;
      c.cls[0] = 0;
      c.coefD[0] = sa[s] / (ma * ma);
      c.coefK[0] = sa[s] / ma;
    } else {
      c.n_terms = S;
      for (int t = 0; t < S; ++t) {
        c.cls[t] = t;
        c.coefD[t] = ctx->nu[s * S + t] / (ma * ma);
        c.coefK[t] = ctx->nu[s * S + t] / ma;
      }
    }
  }
  const Combine3* dc;
  if (int rc = upload(ctx, comb, &dc)) return rc;
  ctx->d_comb = const_cast<Combine3*>(dc);
  std::vector<Spec3> specs(S);
  for (int s = 0; s < S; ++s) {
    specs[s] = Spec3{ctx->species[s].grid, ctx->dk_off[s], ctx->em_off[s], ctx->v_off[s]};
    ctx->max_cells = std::max(ctx->max_cells, ctx->hg[ctx->species[s].grid].n_cells);
    ctx->max_nnz = std::max(ctx->max_nnz, ctx->hg[ctx->species[s].grid].nnz);
  }
  const Spec3* dsp;
  const DevGrid3* dgr;
  if (int rc = upload(ctx, specs, &dsp)) return rc;
  if (int rc = upload(ctx, ctx->dg, &dgr)) return rc;
  ctx->d_spec = const_cast<Spec3*>(dsp);
  ctx->d_grids = const_cast<DevGrid3*>(dgr);
  // batched solve: pattern views per grid, block offsets per species
  std::vector<landau::SolverGridView> gv(ctx->G);
  for (int g = 0; g < ctx->G; ++g)
    gv[g] = landau::SolverGridView{ctx->hg[g].n_dof, ctx->hg[g].nnz, ctx->d_rowptr[g], ctx->d_colidx[g], ctx->hg[g].diag.data()};
  std::vector<landau::SolverSpeciesView> sv(S);
  for (int s = 0; s < S; ++s) sv[s] = landau::SolverSpeciesView{ctx->species[s].grid, ctx->f_off[s], ctx->v_off[s]};
  if (int rc = landau::solver_create(ctx->solver, ctx->device, gv, sv, ctx->f_stride, ctx->v_stride))
    return fail(ctx, rc, ctx->solver.err);
  return LANDAU_OK;
}

int check_call(landau3v_ctx* ctx, const void* in, int batch, const void* out) {
  if (!ctx) return LANDAU_INVALID_ARG;
  if (batch < 0) return fail(ctx, LANDAU_INVALID_ARG, "negative batch");
  if (batch > 0 && (!in || !out)) return fail(ctx, LANDAU_INVALID_ARG, "null buffer");
  if (ctx->device < 0) return fail(ctx, LANDAU_CUDA_ERROR, "host-only context (cuda_device < 0): no compute, no CPU fallback");
  CUDA_TRY3(ctx, cudaSetDevice(ctx->device));
  return LANDAU_OK;
}

// a1, a2, a2b for entries [b0, b0 + nbc): leaves D, K in ctx->DK
int run_coefficients(landau3v_ctx* ctx, const double* batch_f, int b0, int nbc, cudaStream_t st) {
  const int G = ctx->G, S = ctx->S, NCL = ctx->n_classes;
  // the MMA kernel wins at every batch size (one entry: 0.87 against 1.36 ms on the paper's grids, its 8-column tile mostly
  // padding); the scalar kernel stays as the plain variant for A/B and parity
  const int kern = ctx->inner_kernel ? std::min(ctx->inner_kernel, 2) : 2;
  // DMMA kernel, stream mode: persistent CTAs share the (item, source tile) steps evenly -- one plane of G, no wave tail
  bool stream = false;
  StreamPlan3 spl;
  int stream_ctas = 0;
  if (kern == 2 && ctx->inner_kernel != 3 && (nbc > 8 || ctx->inner_kernel == 2)) {  // 8 columns: the grid is as fast and K2b cheap
    const int nt = inner_dmma_nt(nbc);
    if (ctx->dmma_stream_ctas_per_sm[nt] == 0) ctx->dmma_stream_ctas_per_sm[nt] = inner_dmma_stream_ctas_per_sm(nt);
    stream_ctas = ctx->dmma_stream_ctas_per_sm[nt] * ctx->n_sm;
    spl = inner_dmma_stream_plan(ctx->n_pad, ctx->ranges, NCL, nbc);
    stream = spl.step0[NCL] >= stream_ctas;
    for (int c = 0; c < NCL; ++c) stream = stream && spl.njt[c] > 0;
    if (stream)
      if (int rc = grow(ctx, &ctx->part_buf, &ctx->part_cap, inner_dmma_stream_scratch(nt, stream_ctas, spl))) return rc;
  }
  // grid mode: cut the source range when (field tiles x column tiles) alone do not give four CTAs per SM
  int nsplit = 1;
  if (kern == 2 && !stream) {
    const int ncol = nbc > 16 ? 32 : nbc > 8 ? 16 : 8;
    const long long items = (long long)(ctx->n_pad / (K2D_WARPS * 8)) * NCL * ((nbc + ncol - 1) / ncol);
    int min_tiles = 1 << 30;
    for (int c = 0; c < NCL; ++c) min_tiles = std::min(min_tiles, (ctx->ranges.j1[c] - ctx->ranges.j0[c]) / K2D_TJ);
    const int nt = inner_dmma_nt(nbc);
    if (ctx->dmma_ctas_per_sm[nt] == 0) ctx->dmma_ctas_per_sm[nt] = inner_dmma_ctas_per_sm(nt);
    nsplit = inner_dmma_split(items, (long long)ctx->dmma_ctas_per_sm[nt] * ctx->n_sm, std::max(1, std::min(min_tiles / 4, 32)));
  }
  const long long split_stride = (long long)NCL * nbc * 9 * ctx->n_pad;
  const size_t f_need = (size_t)NCL * nbc * 4 * ctx->n_pad, g_need = (size_t)split_stride * nsplit;
  {
    const size_t cap0 = ctx->F_cap;
    if (int rc = grow(ctx, &ctx->F, &ctx->F_cap, f_need)) return rc;
    // entries of F that no kernel writes (padding points, other grids' ranges of a species column) must read as zero
    if (cap0 != ctx->F_cap || ctx->f_nbc != nbc) CUDA_TRY3(ctx, cudaMemsetAsync(ctx->F, 0, f_need * sizeof(double), st));
    ctx->f_nbc = nbc;
  }
  if (int rc = grow(ctx, &ctx->Gs, &ctx->G_cap, g_need)) return rc;
  if (int rc = grow(ctx, &ctx->DK, &ctx->DK_cap, (size_t)ctx->dk_stride * nbc)) return rc;
  mark(ctx, st);
  nvtxRangePushA("landau3v K1 fields (a1)");
  for (int g = 0; g < G; ++g) {
    if (!ctx->mix[g].n_entries) continue;
    k3v_fields<<<dim3(ctx->hg[g].n_cells, nbc), 32, 0, st>>>(ctx->dg[g], ctx->d_tab, ctx->mix[g], batch_f, ctx->f_stride, b0,
                                                             nbc, ctx->F, ctx->n_pad);
    ++ctx->launches;
  }
  nvtxRangePop();
  mark(ctx, st);
  nvtxRangePushA("landau3v K2 inner integral (a2)");
  if (kern == 2 && stream) {
    if (launch_inner_dmma_stream(ctx->d_px, ctx->d_py, ctx->d_pz, ctx->n_pad, ctx->ranges, nbc, spl, stream_ctas, ctx->F, ctx->Gs,
                                 ctx->part_buf, st)) {
      nvtxRangePop();
      return fail(ctx, LANDAU_CUDA_ERROR, "k3v_inner_dmma_stream launch failed");
    }
    ++ctx->launches;  // the counter memset
  } else if (kern == 2) {
    if (int rc = launch_inner_dmma(ctx->d_px, ctx->d_py, ctx->d_pz, ctx->n_pad, ctx->ranges, NCL, nbc, nsplit, ctx->F, ctx->Gs, split_stride, st)) {
      nvtxRangePop();
      return fail(ctx, rc, "k3v_inner_dmma launch configuration failed");
    }
  } else {
    if (nbc >= 4)
      k3v_inner_dfma<4><<<dim3(ctx->n_pad / K2_TI, NCL * ((nbc + 3) / 4)), K2_TI, 0, st>>>(ctx->d_px, ctx->d_py, ctx->d_pz, ctx->n_pad,
                                                                                         ctx->ranges, nbc, ctx->F, ctx->Gs);
    else if (nbc >= 2)
      k3v_inner_dfma<2><<<dim3(ctx->n_pad / K2_TI, NCL * ((nbc + 1) / 2)), K2_TI, 0, st>>>(ctx->d_px, ctx->d_py, ctx->d_pz, ctx->n_pad,
                                                                                         ctx->ranges, nbc, ctx->F, ctx->Gs);
    else
      k3v_inner_dfma<1><<<dim3(ctx->n_pad / K2_TI, NCL * nbc), K2_TI, 0, st>>>(ctx->d_px, ctx->d_py, ctx->d_pz, ctx->n_pad,
                                                                             ctx->ranges, nbc, ctx->F, ctx->Gs);
  }
  ++ctx->launches;
  nvtxRangePop();
  mark(ctx, st);
  nvtxRangePushA("landau3v K2b combine (a2)");
  k3v_combine<<<dim3((ctx->max_ip + 255) / 256, nbc, S), 256, 0, st>>>(ctx->d_comb, ctx->Gs, ctx->n_pad, nbc, nsplit, split_stride, ctx->DK,
                                                                       ctx->dk_stride);
  ++ctx->launches;
  nvtxRangePop();
  mark(ctx, st);
  CUDA_TRY3(ctx, cudaGetLastError());
  return LANDAU_OK;
}

int assemble_chunk(landau3v_ctx* ctx, int b0, int nbc, double inv_dt, double* out, cudaStream_t st) {
  nvtxRangePushA("landau3v K3 element matrices + assembly (a3+a4)");
  double* vals = out + (long long)b0 * ctx->v_stride;
  if (ctx->assembly_kernel == 1) {
    for (int s = 0; s < ctx->S; ++s) {
      const int g = ctx->species[s].grid;
      k3v_assemble<<<dim3((ctx->hg[g].nnz + 127) / 128, nbc), 128, 0, st>>>(ctx->dg[g], ctx->d_tab, ctx->DK, ctx->dk_stride,
                                                                            ctx->dk_off[s], inv_dt, vals, ctx->v_stride, ctx->v_off[s]);
      ++ctx->launches;
    }
  } else {
    if (int rc = grow(ctx, &ctx->EM, &ctx->EM_cap, (size_t)ctx->em_stride * nbc)) {
      nvtxRangePop();
      return rc;
    }
    if (!ctx->k3e_configured) {
      cudaFuncSetAttribute(k3v_elem_matrix, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)K3E_SMEM);
      ctx->k3e_configured = true;
    }
    {
      if (ctx->k3e_ctas_per_sm == 0) {
        int n = 0;
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k3v_elem_matrix, K3E_WARPS * 32, K3E_SMEM);
        ctx->k3e_ctas_per_sm = n > 0 ? n : 1;
      }
      const long long items = (long long)ctx->S * nbc * ctx->max_cells;
      const int grid = (int)std::max(1LL, std::min<long long>((items + K3E_WARPS - 1) / K3E_WARPS, (long long)ctx->k3e_ctas_per_sm * ctx->n_sm));
      k3v_elem_matrix<<<grid, K3E_WARPS * 32, K3E_SMEM, st>>>(ctx->d_grids, ctx->d_spec, ctx->S, nbc, ctx->max_cells, ctx->d_tab, ctx->DK,
                                                              ctx->dk_stride, inv_dt, ctx->EM, ctx->em_stride);
    }
    k3v_gather<<<dim3((ctx->max_nnz + 255) / 256, (nbc + K3G_BT - 1) / K3G_BT, ctx->S), 256, 0, st>>>(
        ctx->d_grids, ctx->d_spec, nbc, ctx->EM, ctx->em_stride, vals, ctx->v_stride);
    ctx->launches += 2;
  }
  nvtxRangePop();
  return LANDAU_OK;
}

int apply_chunk(landau3v_ctx* ctx, const double* batch_f, int b0, int nbc, double* out_rhs, cudaStream_t st) {
  if (int rc = grow(ctx, &ctx->FE, &ctx->FE_cap, (size_t)ctx->fe_stride * nbc)) return rc;
  nvtxRangePushA("landau3v K3' apply (a5)");
  for (int s = 0; s < ctx->S; ++s) {
    const int g = ctx->species[s].grid;
    k3v_elem_apply<<<dim3(ctx->hg[g].n_cells, nbc), 32, 0, st>>>(ctx->dg[g], ctx->d_tab, batch_f, ctx->f_stride, ctx->f_off[s], b0, ctx->DK,
                                                                 ctx->dk_stride, ctx->dk_off[s], ctx->FE, ctx->fe_stride, ctx->fe_off[s]);
    k3v_apply_gather<<<dim3((ctx->hg[g].n_dof + 127) / 128, nbc), 128, 0, st>>>(ctx->dg[g], ctx->FE, ctx->fe_stride, ctx->fe_off[s], out_rhs,
                                                                                ctx->f_stride, ctx->f_off[s], b0);
    ctx->launches += 2;
  }
  nvtxRangePop();
  return LANDAU_OK;
}

}  // namespace

extern "C" {

int landau3v_create(const landau3v_grid_desc* grids, int n_grids, const landau_species_desc* species, int n_species,
                    const double* nu, int cuda_device, landau3v_ctx** out) {
  if (!grids || !species || !out || n_grids < 1 || n_species < 1)
    return fail(nullptr, LANDAU_INVALID_ARG, "null argument or empty grid/species list");
  if (n_species > MAX_TERMS) return fail(nullptr, LANDAU_UNSUPPORTED, "at most 16 species");
  landau3v_ctx* ctx = new (std::nothrow) landau3v_ctx();
  if (!ctx) return fail(nullptr, LANDAU_OUT_OF_MEMORY, "host allocation failed");
  auto bail = [&](int code, const std::string& m) {
    landau3v_destroy(ctx);
    return fail(nullptr, code, m);
  };
  try {
    build_tables3(&ctx->ht);
    ctx->G = n_grids;
    ctx->S = n_species;
    ctx->hg.resize(n_grids);
    std::string msg;
    ctx->ip_off.assign(n_grids + 1, 0);
    for (int g = 0; g < n_grids; ++g) {
      if (int rc = build_grid3(grids[g], ctx->ht, &ctx->hg[g], &msg)) return bail(rc, msg);
      ctx->ip_off[g + 1] = ctx->ip_off[g] + ctx->hg[g].n_ip;
      ctx->max_ip = std::max(ctx->max_ip, ctx->hg[g].n_ip);
    }
    ctx->n_ip_total = ctx->ip_off[n_grids];
    ctx->species.assign(species, species + n_species);
    ctx->nu.resize((size_t)n_species * n_species);
    long long fo = 0, vo = 0, dko = 0, feo = 0;
    for (int a = 0; a < n_species; ++a) {
      if (species[a].grid < 0 || species[a].grid >= n_grids || !(species[a].mass > 0))
        return bail(LANDAU_INVALID_ARG, "species with bad grid index or mass");
      for (int b = 0; b < n_species; ++b)
        ctx->nu[a * n_species + b] = nu ? nu[a * n_species + b]
                                        : species[a].charge * species[a].charge * species[b].charge * species[b].charge;
      const HostGrid3& h = ctx->hg[species[a].grid];
      ctx->f_off.push_back(fo);
      ctx->v_off.push_back(vo);
      ctx->dk_off.push_back(dko);
      ctx->fe_off.push_back(feo);
      ctx->em_off.push_back(feo * NB);
      fo += h.n_dof;
      vo += h.nnz;
      dko += 9LL * h.n_ip;
      feo += (long long)h.n_cells * NB;
    }
    ctx->f_stride = fo;
    ctx->v_stride = vo;
    ctx->dk_stride = dko;
    ctx->fe_stride = feo;
    ctx->em_stride = feo * NB;
  } catch (const std::bad_alloc&) {
    return bail(LANDAU_OUT_OF_MEMORY, "host allocation failed");
  }
  ctx->device = cuda_device;
  if (cuda_device < 0) {
    *out = ctx;
    return LANDAU_OK;
  }
  cudaError_t e = cudaSetDevice(cuda_device);
  if (e != cudaSuccess) return bail(LANDAU_CUDA_ERROR, std::string("cudaSetDevice: ") + cudaGetErrorString(e));
  cudaDeviceGetAttribute(&ctx->n_sm, cudaDevAttrMultiProcessorCount, cuda_device);
  if (int rc = build_device_side(ctx)) {
    const std::string m = ctx->err;
    return bail(rc, m);
  }
  *out = ctx;
  return LANDAU_OK;
}

void landau3v_destroy(landau3v_ctx* ctx) {
  if (!ctx) return;
  if (ctx->device >= 0 && !ctx->allocs.empty()) {
    cudaSetDevice(ctx->device);
    cudaDeviceSynchronize();
  }
  for (void* p : ctx->allocs) cudaFree(p);
  landau::solver_destroy(ctx->solver);
  for (double* p : {ctx->F, ctx->Gs, ctx->DK, ctx->FE, ctx->EM, ctx->stage_in, ctx->stage_out, ctx->st_M, ctx->part_buf})
    if (p) cudaFree(p);
  for (cudaEvent_t e : ctx->ev) cudaEventDestroy(e);
  delete ctx;
}

int landau3v_sizes(const landau3v_ctx* ctx, int* n_dof, int* nnz, int* n_ip, int* n_cells, long long* f_stride,
                   long long* csr_stride) {
  if (!ctx) return LANDAU_INVALID_ARG;
  for (int g = 0; g < ctx->G; ++g) {
    if (n_dof) n_dof[g] = ctx->hg[g].n_dof;
    if (nnz) nnz[g] = ctx->hg[g].nnz;
    if (n_ip) n_ip[g] = ctx->hg[g].n_ip;
    if (n_cells) n_cells[g] = ctx->hg[g].n_cells;
  }
  if (f_stride) *f_stride = ctx->f_stride;
  if (csr_stride) *csr_stride = ctx->v_stride;
  return LANDAU_OK;
}

int landau3v_dof_coords(const landau3v_ctx* ctx, int grid, double* xyz_host) {
  if (!ctx || !xyz_host || grid < 0 || grid >= ctx->G) return LANDAU_INVALID_ARG;
  memcpy(xyz_host, ctx->hg[grid].dof_xyz.data(), sizeof(double) * ctx->hg[grid].dof_xyz.size());
  return LANDAU_OK;
}

int landau3v_ip_table(const landau3v_ctx* ctx, int grid, double* x, double* y, double* z, double* w) {
  if (!ctx || grid < 0 || grid >= ctx->G) return LANDAU_INVALID_ARG;
  const HostGrid3& h = ctx->hg[grid];
  if (x) memcpy(x, h.ip_x.data(), sizeof(double) * h.n_ip);
  if (y) memcpy(y, h.ip_y.data(), sizeof(double) * h.n_ip);
  if (z) memcpy(z, h.ip_z.data(), sizeof(double) * h.n_ip);
  if (w) memcpy(w, h.ip_w.data(), sizeof(double) * h.n_ip);
  return LANDAU_OK;
}

int landau3v_csr_pattern(const landau3v_ctx* ctx, int grid, const int** rowptr_dev, const int** colidx_dev) {
  if (!ctx || grid < 0 || grid >= ctx->G || !rowptr_dev || !colidx_dev || ctx->device < 0) return LANDAU_INVALID_ARG;
  *rowptr_dev = ctx->d_rowptr[grid];
  *colidx_dev = ctx->d_colidx[grid];
  return LANDAU_OK;
}

int landau3v_csr_pattern_host(const landau3v_ctx* ctx, int grid, int* rowptr_host, int* colidx_host) {
  if (!ctx || grid < 0 || grid >= ctx->G || !rowptr_host || !colidx_host) return LANDAU_INVALID_ARG;
  const HostGrid3& h = ctx->hg[grid];
  memcpy(rowptr_host, h.rowptr.data(), sizeof(int) * h.rowptr.size());
  memcpy(colidx_host, h.colidx.data(), sizeof(int) * h.colidx.size());
  return LANDAU_OK;
}

int landau3v_jacobian(landau3v_ctx* ctx, const double* batch_f_dev, int batch, double dt, double* out_csr_vals_dev,
                      void* cuda_stream) {
  if (int rc = check_call(ctx, batch_f_dev, batch, out_csr_vals_dev)) return rc;
  if (!(dt > 0)) return fail(ctx, LANDAU_INVALID_ARG, "dt must be > 0 (use +inf for the unshifted -J)");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const double inv_dt = std::isinf(dt) ? 0.0 : 1.0 / dt;
  ctx->ev_used = 0;
  for (int b0 = 0; b0 < batch; b0 += ctx->chunk) {
    const int nbc = std::min(ctx->chunk, batch - b0);
    if (int rc = run_coefficients(ctx, batch_f_dev, b0, nbc, st)) return rc;
    if (int rc = assemble_chunk(ctx, b0, nbc, inv_dt, out_csr_vals_dev, st)) return rc;
    CUDA_TRY3(ctx, cudaGetLastError());
    mark(ctx, st);
    ctx->last_batch = nbc;
  }
  ctx->last_stream = st;
  return LANDAU_OK;
}

int landau3v_apply(landau3v_ctx* ctx, const double* batch_f_dev, int batch, double* out_rhs_dev, void* cuda_stream) {
  if (int rc = check_call(ctx, batch_f_dev, batch, out_rhs_dev)) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  ctx->ev_used = 0;
  for (int b0 = 0; b0 < batch; b0 += ctx->chunk) {
    const int nbc = std::min(ctx->chunk, batch - b0);
    if (int rc = run_coefficients(ctx, batch_f_dev, b0, nbc, st)) return rc;
    if (int rc = apply_chunk(ctx, batch_f_dev, b0, nbc, out_rhs_dev, st)) return rc;
    CUDA_TRY3(ctx, cudaGetLastError());
    mark(ctx, st);
    ctx->last_batch = nbc;
  }
  ctx->last_stream = st;
  return LANDAU_OK;
}

int landau3v_jacobian_apply(landau3v_ctx* ctx, const double* batch_f_dev, int batch, double dt, double* out_csr_vals_dev,
                            double* out_rhs_dev, void* cuda_stream) {
  if (int rc = check_call(ctx, batch_f_dev, batch, out_csr_vals_dev)) return rc;
  if (batch > 0 && !out_rhs_dev) return fail(ctx, LANDAU_INVALID_ARG, "null buffer");
  if (!(dt > 0)) return fail(ctx, LANDAU_INVALID_ARG, "dt must be > 0 (use +inf for the unshifted -J)");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const double inv_dt = std::isinf(dt) ? 0.0 : 1.0 / dt;
  ctx->ev_used = 0;
  for (int b0 = 0; b0 < batch; b0 += ctx->chunk) {
    const int nbc = std::min(ctx->chunk, batch - b0);
    if (int rc = run_coefficients(ctx, batch_f_dev, b0, nbc, st)) return rc;
    if (int rc = assemble_chunk(ctx, b0, nbc, inv_dt, out_csr_vals_dev, st)) return rc;
    if (int rc = apply_chunk(ctx, batch_f_dev, b0, nbc, out_rhs_dev, st)) return rc;
    CUDA_TRY3(ctx, cudaGetLastError());
    mark(ctx, st);
    ctx->last_batch = nbc;
  }
  ctx->last_stream = st;
  return LANDAU_OK;
}

int landau3v_spmv(landau3v_ctx* ctx, const double* csr_vals_dev, const double* x_dev, int batch, double* y_dev,
                  void* cuda_stream) {
  if (int rc = check_call(ctx, csr_vals_dev, batch, y_dev)) return rc;
  if (batch > 0 && !x_dev) return fail(ctx, LANDAU_INVALID_ARG, "null buffer");
  if (batch == 0) return LANDAU_OK;
  if (int rc = landau::solver_spmv(ctx->solver, csr_vals_dev, ctx->v_stride, x_dev, batch, y_dev, (cudaStream_t)cuda_stream))
    return fail(ctx, rc, ctx->solver.err);
  return LANDAU_OK;
}

int landau3v_solve(landau3v_ctx* ctx, const double* csr_vals_dev, const double* rhs_dev, int batch, double rtol, int max_it,
                   double* x_dev, int* iters_dev, double* relres_dev, void* cuda_stream) {
  if (int rc = check_call(ctx, csr_vals_dev, batch, x_dev)) return rc;
  if (batch > 0 && !rhs_dev) return fail(ctx, LANDAU_INVALID_ARG, "null buffer");
  if (!(rtol > 0) || max_it < 1) return fail(ctx, LANDAU_INVALID_ARG, "rtol must be > 0 and max_it >= 1");
  if (batch == 0) return LANDAU_OK;
  if (int rc = landau::solver_tfqmr(ctx->solver, csr_vals_dev, rhs_dev, batch, rtol, max_it, x_dev, iters_dev, relres_dev,
                                    (cudaStream_t)cuda_stream))
    return fail(ctx, rc, ctx->solver.err);
  return LANDAU_OK;
}

int landau3v_step(landau3v_ctx* ctx, double* u_dev, int batch, double dt, double newton_rtol, int max_newton,
                  double lin_rtol, int lin_max_it, double* info_host, void* cuda_stream) {
  if (int rc = check_call(ctx, u_dev, batch, u_dev)) return rc;
  if (!(dt > 0) || std::isinf(dt) || max_newton < 1 || !(lin_rtol > 0) || lin_max_it < 1)
    return fail(ctx, LANDAU_INVALID_ARG, "landau3v_step: dt finite > 0, max_newton >= 1, lin_rtol > 0, lin_max_it >= 1");
  if (info_host) info_host[0] = info_host[1] = info_host[2] = info_host[3] = 0.0;
  if (batch == 0) return LANDAU_OK;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  // mass values (independent of f and of the entry): M = (M/1 - J[0]) since D = K = 0 for f = 0
  if (!ctx->st_M) {
    if (int rc = grow(ctx, &ctx->st_M, &ctx->st_M_cap, (size_t)ctx->v_stride + ctx->f_stride)) return rc;
    double* zero_f = ctx->st_M + ctx->v_stride;
    CUDA_TRY3(ctx, cudaMemsetAsync(zero_f, 0, sizeof(double) * ctx->f_stride, st));
    const bool timing = ctx->timing;
    ctx->timing = false;
    const int rc = landau3v_jacobian(ctx, zero_f, 1, 1.0, ctx->st_M, cuda_stream);
    ctx->timing = timing;
    if (rc) return rc;
  }
  const landau::JacobianApplyFn jac = [&](const double* u, int nb, double step, double* A, double* ju) {
    return landau3v_jacobian_apply(ctx, u, nb, step, A, ju, cuda_stream);
  };
  if (int rc = landau::solver_step(ctx->solver, jac, ctx->st_M, u_dev, batch, dt, newton_rtol, max_newton, lin_rtol, lin_max_it,
                                   info_host, st))
    return ctx->solver.err.empty() ? rc : fail(ctx, rc, ctx->solver.err);
  return LANDAU_OK;
}

int landau3v_jacobian_host(landau3v_ctx* ctx, const double* batch_f_host, int batch, double dt, double* out_csr_vals_host,
                           void* cuda_stream) {
  if (int rc = check_call(ctx, batch_f_host, batch, out_csr_vals_host)) return rc;
  if (batch == 0) return LANDAU_OK;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t nin = (size_t)batch * ctx->f_stride, nout = (size_t)batch * ctx->v_stride;
  if (int rc = grow(ctx, &ctx->stage_in, &ctx->stage_in_cap, nin)) return rc;
  if (int rc = grow(ctx, &ctx->stage_out, &ctx->stage_out_cap, nout)) return rc;
  CUDA_TRY3(ctx, cudaMemcpyAsync(ctx->stage_in, batch_f_host, nin * sizeof(double), cudaMemcpyHostToDevice, st));
  if (int rc = landau3v_jacobian(ctx, ctx->stage_in, batch, dt, ctx->stage_out, cuda_stream)) return rc;
  CUDA_TRY3(ctx, cudaMemcpyAsync(out_csr_vals_host, ctx->stage_out, nout * sizeof(double), cudaMemcpyDeviceToHost, st));
  CUDA_TRY3(ctx, cudaStreamSynchronize(st));
  return LANDAU_OK;
}

int landau3v_last_coefficients(landau3v_ctx* ctx, double* dk_host, int n_entries) {
  if (!ctx || !dk_host || n_entries < 1) return LANDAU_INVALID_ARG;
  if (ctx->device < 0 || ctx->last_batch == 0 || !ctx->DK) return fail(ctx, LANDAU_INVALID_ARG, "no previous jacobian/apply call");
  if (n_entries > ctx->last_batch) return fail(ctx, LANDAU_INVALID_ARG, "landau3v_last_coefficients: more entries asked than the last pass holds");
  CUDA_TRY3(ctx, cudaSetDevice(ctx->device));
  CUDA_TRY3(ctx, cudaStreamSynchronize(ctx->last_stream));
  CUDA_TRY3(ctx, cudaMemcpy(dk_host, ctx->DK, sizeof(double) * ctx->dk_stride * n_entries, cudaMemcpyDeviceToHost));
  return LANDAU_OK;
}

int landau3v_set_timing(landau3v_ctx* ctx, int enabled) {
  if (!ctx) return LANDAU_INVALID_ARG;
  ctx->timing = enabled != 0;
  return LANDAU_OK;
}

int landau3v_last_stage_ms(landau3v_ctx* ctx, float* ms4) {
  if (!ctx || !ms4) return LANDAU_INVALID_ARG;
  for (int k = 0; k < 4; ++k) ms4[k] = 0;
  if (ctx->ev_used >= 5) {
    CUDA_TRY3(ctx, cudaEventSynchronize(ctx->ev[ctx->ev_used - 1]));
    for (int p = 0; p + 5 <= ctx->ev_used; p += 5)
      for (int k = 0; k < 4; ++k) {
        float ms = 0;
        cudaEventElapsedTime(&ms, ctx->ev[p + k], ctx->ev[p + k + 1]);
        ms4[k] += ms;
      }
  }
  return LANDAU_OK;
}

long long landau3v_launch_count(const landau3v_ctx* ctx) { return ctx ? ctx->launches + ctx->solver.launches : 0; }

int landau3v_set_inner_kernel(landau3v_ctx* ctx, int which) {
  if (!ctx || which < 0 || which > 3) return LANDAU_INVALID_ARG;
  ctx->inner_kernel = which;
  return LANDAU_OK;
}

int landau3v_set_assembly_kernel(landau3v_ctx* ctx, int which) {
  if (!ctx || which < 0 || which > 1) return LANDAU_INVALID_ARG;
  ctx->assembly_kernel = which;
  return LANDAU_OK;
}

int landau3v_set_batch_chunk(landau3v_ctx* ctx, int chunk) {
  if (!ctx || chunk < 1) return LANDAU_INVALID_ARG;
  ctx->chunk = chunk;
  return LANDAU_OK;
}

const char* landau3v_last_error(const landau3v_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_error3.c_str(); }

}  // extern "C"
