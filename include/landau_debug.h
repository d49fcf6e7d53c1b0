/* landau_debug.h -- diagnostics, probes and tuning knobs of liblandau_b200.so.
 *
 * NOT part of the product ABI (include/landau.h): these entry points exist for the test-suite (pieces of the path
 * checked alone against the oracle), for bench.py (stage timings, roofline denominators, launch counts) and for
 * kernel A/B measurements.  Same conventions as landau.h (plain C, "host"/"dev" says where memory lives, return 0 or a
 * negative landau_status).  They may change between rounds.
 */
#ifndef LANDAU_B200_DEBUG_H
#define LANDAU_B200_DEBUG_H

#include "landau.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Copy out the frozen coefficients of the LAST landau_jacobian / landau_apply call (synchronises the stream it
 * ran on): dk_host[n_entries][species a][5][n_ip[grid(a)]] = (Drr, Drz, Dzz, Kr, Kz) at the integration points
 * (eq. 2.3).  Only the last pass (batch chunk) of the call is kept:
 * n_entries must be between 1 and the number of entries of that pass, else LANDAU_INVALID_ARG (nothing is copied). */
int landau_last_coefficients(landau_ctx* ctx, double* dk_host, int n_entries);

/* Evaluate the 2V Landau tensor kernel on the device for n point pairs (dev arrays r,z,rb,zb of n doubles):
 * out_dev[5*n] = (UD_rr, UD_rz, UD_zz, UK_rr, UK_zr) per pair, UK_rz = UD_rz, UK_zz = UD_zz; coincident
 * pairs give zeros.  Same device function as the inner-integral kernel uses. */
int landau_tensor_eval(const double* r_dev, const double* z_dev, const double* rb_dev, const double* zb_dev, int n,
                       double* out_dev, void* cuda_stream);

/* Elliptic pieces on the device: for n pairs (m[i], mp[i] = 1-m[i] given separately) out_dev[3*n] =
 * (P0, Dc, Q) = INT_0^{pi/2} {1, cos^2, sin^2 cos^2} (1 - m sin^2)^{-3/2} dtheta. */
int landau_ellip_eval(const double* m_dev, const double* mp_dev, int n, double* out_dev, void* cuda_stream);

/* FP64 pipe probes used by bench.py for the roofline denominator: run `iters` rounds of register-resident
 * DFMA (kind 0), DMMA m8n8k4 (kind 1) or both interleaved (kind 2) on every SM; *tflops receives the achieved FP64 TFLOP/s
 * (CUDA-event timed on `cuda_stream`, synchronises it). */
int landau_fp64_probe(int kind, int iters, double* tflops, void* cuda_stream);

/* L2 read-bandwidth probe, the roofline denominator of the batched solve on systems whose matrix values stream from L2 (the
 * guides give no L2 figure): every thread block reads a buffer of `bytes` (1 MiB .. 1 GiB; choose one that stays L2-resident,
 * e.g. 32 MiB) `iters` times with 16-byte L1-bypassing loads; *gbs receives bytes * iters / time in GB/s, best of three timed
 * launches after one that warms the cache.  Allocates and frees its buffer; synchronises `cuda_stream`. */
int landau_l2_probe(long long bytes, int iters, double* gbs, void* cuda_stream);

/* 1 if the collision-frequency matrix was detected as rank one (nu_ab = a_a b_b: one summed source column per
 * batch entry), 0 if the general per-species-column path is used; negative on error. */
int landau_is_separable(const landau_ctx* ctx);

/* Number of kernels the library launched on behalf of this context since creation (bench's gpu_launches). */
long long landau_launch_count(const landau_ctx* ctx);

/* Per-stage device time of the LAST jacobian/apply call in milliseconds, summed over its passes: ms[0] field
 * evaluation, ms[1] inner integral, ms[2] coefficient combination, ms[3] element matrices + assembly (or apply).
 * Recording is enabled with landau_set_timing(ctx, 1): the compute calls then only RECORD CUDA events on their
 * stream (no synchronisation is added to them); landau_last_stage_ms waits for the last event and reads them. */
int landau_set_timing(landau_ctx* ctx, int enabled);
int landau_last_stage_ms(landau_ctx* ctx, float* ms4);

/* Choose the inner-integral kernel: 0 auto (by column count), 1 plain DFMA kernel, 2 DMMA kernel with per-warp
 * tensor generation, 3 / 4 DMMA GEMM kernel with the tensor tile evaluated once per CTA and shared by its warps
 * (TMA-staged source tiles; 16 x 128 / 16 x 256 CTA tile: defaults for 65 .. 128 and for more than 128 source columns), 5 the
 * same with a 16 x 64 tile (default for 49 .. 64 columns).  The three run as persistent CTAs that cut the tiles of the last
 * partial wave along the source range whenever the tile count is not a multiple of the resident CTAs. */
int landau_set_inner_kernel(landau_ctx* ctx, int which);

/* Choose the element-matrix + assembly kernel: 0 auto (k3_ring: DMMA sum-factorised element matrices kept in a
 * shared-memory ring, CSR slots gathered from it; used for every grid whose ring fits in shared memory -- the other grids,
 * e.g. triangles, take k3_elem_matrix + k3_gather: element matrices to a scratch array, then one gather per CSR slot),
 * 1 force the first general kernel (k3_assemble: one thread per CSR slot integrating its own entries, scalar FP64), 2 the ring
 * kernel without the tail cut (one CTA per (entry, species) block), 3 element matrices + gather for every grid (1 - 3: for A/B
 * measurements and parity tests). */
int landau_set_assembly_kernel(landau_ctx* ctx, int which);

/* Choose the launch mode of the batched TFQMR solve: 0 / 1 one thread block per system (default), 2 ONE WARP per system
 * where at least four systems fit in the shared memory of an SM with their values and vectors (e.g. the 142-unknown blocks
 * of the paper's 2V throughput problem): the warps of a thread block take entries of one species and share its pattern, no
 * block-wide barrier in the iteration.  Same iterates; measured SLOWER (1.48 against 1.31 ms for 2560 systems: six warps per
 * SM hide less latency than sixteen), kept for A/B measurements only. */
int landau_set_solve_kernel(landau_ctx* ctx, int which);

/* What landau_solve will launch on this context under the current knob: warps_per_block > 0 (4..8) when the next solve
 * runs the warp-per-system kernel with that many systems per thread block, 0 when it runs one thread block per system
 * (the default, and what mode 2 silently falls back to when four systems do not fit in an SM's shared memory).  Lets a
 * test assert that the kernel it means to exercise is the one that runs.  Host query; either pointer may be NULL.
 *   max_unknowns     : largest n_dof over the context's grids (the size the shared-memory plan is made for)
 *   matrix_in_shared : 1 when every system's CSR values and pattern are copied to shared memory once and the products of
 *                      the iteration run from there (small systems); 0 when they stream from L2 in every product. */
int landau_solve_mode(const landau_ctx* ctx, int* warps_per_block, int* max_unknowns, int* matrix_in_shared);

/* Schedule of the ring assembly kernel for grid g (host query, works on host-only contexts): ring_cells = element
 * matrices kept in shared memory (0: the ring does not fit, the slot-gather kernel is used for this grid),
 * n_steps = panels of 8 cells, n_simple_slots = CSR slots fed by exactly one element-matrix entry with weight 1. */
int landau_assembly_info(const landau_ctx* ctx, int grid, int* ring_cells, int* n_steps, int* n_simple_slots);

/* Batch entries pushed through the stages per pass (default 1024); scratch is sized for one pass, so that the
 * intermediates (source fields, partial sums, D/K) of a pass stay L2-resident.  chunk >= 1. */
int landau_set_batch_chunk(landau_ctx* ctx, int chunk);

#ifdef __cplusplus
}
#endif
#endif /* LANDAU_B200_DEBUG_H */
