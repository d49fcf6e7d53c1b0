#!/usr/bin/env python
"""bench.py -- throughput of the batched Landau Jacobian construction (BASELINE.json metric) on N B200s.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 5] [--batch 1024] [--impl ours|reference]

One "step" = one pass of the whole hot path (a1 field evaluation, a2 inner integral, a2b species combination,
a3+a4 element matrices + assembly into the batched CSR of M/dt - J) over one batch of seeded synthetic
distribution functions.  Default workload: BASELINE.json configs[4] ("large-batch
throughput ... Jacobian build + assembly timed end to end"), e-/D+ on uniform 14x28 Q3 grids, batch 1024 per GPU
(DESIGN.md "Measurement" says why this one and not configs[1]; `--config 2 --batch 64` runs configs[1]).

Prints ONE JSON line (rank 0): value = Landau Jacobians/s of the whole job, device-resident inputs; e2e = same
metric through landau_jacobian_host (pinned HOST buffers, H2D + D2H inside the timed region); roofline = the
inner-integral kernel (K2) against the FP64 pipe peak measured in-process; cpu_baseline = the oracle, as it
stands, on the host cores over a bounded sample of the same workload.

`--impl reference` times the oracle only (no GPU work); under torchrun only rank 0 runs it.

Extras that do not enter `value`: `--solve` times the batched TFQMR solve of the step's backward-Euler systems
(key "solve"), `--advance N` runs N backward-Euler steps of the batch with landau_step (key "advance": seconds,
Newton iterations, Newton iterations x batch per second -- the paper's throughput measure);
`--config 6` is the paper's own throughput problem.
"""
import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "landau_jacobians_per_s"
UNIT = "Jacobians/s"
FLOP_PER_PAIR_COLUMN = 14.0   # 7 FP64 FMA per (i, j, source column): DESIGN.md "Algorithmic work"
TENSOR_FLOP_PER_PAIR = 250.0  # one evaluation of the 5 tensor components (counted from SASS)


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5, help="BASELINE.json config number 1..5 (6: the paper's throughput problem)")
    ap.add_argument("--batch", type=int, default=None, help="batch entries PER GPU (default: the config's)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="CPU time budget of the cpu_baseline sample")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--kernel", type=int, default=0, help="inner-integral kernel: 0 auto, 1 DFMA, 2 DMMA, 3/4 GEMM (32x128 / 16x256 tile)")
    ap.add_argument("--solve", action="store_true", help="also time the batched TFQMR solve of the step's systems "
                    "(reported under \"solve\", not part of value)")
    ap.add_argument("--advance", type=int, default=0, help="also run this many backward-Euler steps (landau_step) and "
                    "report the time and Newton iterations under \"advance\" (not part of value)")
    ap.add_argument("--assembly", type=int, default=0, help="assembly kernel build (landau_set_assembly_kernel; 0: default)")
    ap.add_argument("--chunk", type=int, default=0, help="batch entries per pass through the stages (0: library default)")
    return ap.parse_args()


def workload_name(cfg, B):
    return "%s batch=%d/GPU (BASELINE.json configs[%d])" % (cfg["name"], B, cfg["index"] - 1)


# ----------------------------------------------------------------------------------------------------------------
# the oracle arm: cpu_baseline leg and --impl reference
# ----------------------------------------------------------------------------------------------------------------
def oracle_sample(cfg, seconds, min_entries=1, max_entries=64):
    """Time the oracle (as it stands, OpenMP over field points) on entries 0, 1, ... of the workload until
    `seconds` of wall time are used.  Returns (Jacobians/s, entries done, threads, per-entry seconds)."""
    from oracle import oracle as O
    from paper_2209_03228_b200 import workloads as W
    O.build()
    o = O.Oracle(cfg["grids"], cfg["species"], cfg["degree"])
    coords = [o.dof_coords(g) for g in range(o.G)]
    times = []
    t_start = time.perf_counter()
    b = 0
    while b < max_entries and (b < min_entries or time.perf_counter() - t_start < seconds):
        f = W.make_batch_f(cfg, coords, entries=[b])[0]
        t0 = time.perf_counter()
        o.jacobian(f, cfg["dt"])
        times.append(time.perf_counter() - t0)
        b += 1
    total = sum(times)
    return len(times) / total, len(times), o.threads, times


def run_reference(args):
    from paper_2209_03228_b200 import workloads as W
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = W.config(args.config)
    B = args.batch or cfg["batch"]
    # a step = a bounded sample: ONE Jacobian (entry s mod B) of the workload on all host cores
    from oracle import oracle as O
    O.build()
    o = O.Oracle(cfg["grids"], cfg["species"], cfg["degree"])
    coords = [o.dof_coords(g) for g in range(o.G)]
    fs = [W.make_batch_f(cfg, coords, entries=[s % B])[0] for s in range(args.steps + args.warmup)]
    for s in range(args.warmup):
        o.jacobian(fs[s], cfg["dt"])
    t0 = time.perf_counter()
    for s in range(args.steps):
        o.jacobian(fs[args.warmup + s], cfg["dt"])
    dt = time.perf_counter() - t0
    value = args.steps / dt
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64 (long double sums)",
            "data": "synthetic", "config": {"workload": workload_name(cfg, B), "sample": "1 Jacobian per step"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": o.threads, "kind": "oracle",
                             "sample": "one Jacobian (one batch entry, all species blocks) of the workload per step"},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------------------------------
# clocks sampler
# ----------------------------------------------------------------------------------------------------------------
class ClockSampler:
    FIELDS = ["clocks.sm", "clocks.max.sm", "power.draw", "clocks_event_reasons.hw_slowdown",
              "clocks_event_reasons.hw_thermal_slowdown", "clocks_event_reasons.sw_thermal_slowdown",
              "clocks_event_reasons.sw_power_cap"]

    def __init__(self, index):
        self.rows = []
        self.proc = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(index), "--query-gpu=" + ",".join(self.FIELDS),
                 "--format=csv,noheader,nounits", "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL,
                text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), [x.strip() for x in line.split(",")]))

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.proc.kill()

    def summary(self, t0, t1):
        sel = [r for (t, r) in self.rows if t0 <= t <= t1 and len(r) == len(self.FIELDS)] or \
              [r for (_, r) in self.rows if len(r) == len(self.FIELDS)]
        if not sel:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        def num(x):
            try:
                return float(x)
            except ValueError:
                return float("nan")
        sm = sorted(num(r[0]) for r in sel)
        reasons = []
        for k, name in enumerate(["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]):
            if any(r[3 + k].lower().startswith("active") for r in sel):
                reasons.append(name)
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": num(sel[0][1]), "power_w_max": max(num(r[2]) for r in sel),
                "reasons": reasons, "samples": len(sel)}


# ----------------------------------------------------------------------------------------------------------------
# our arm
# ----------------------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    from paper_2209_03228_b200 import binding as Bn
    from paper_2209_03228_b200 import sharding
    from paper_2209_03228_b200 import workloads as W

    rank, world, local = sharding.env_rank()
    if world != args.gpus and world > 1:
        raise SystemExit("--gpus %d but WORLD_SIZE=%d" % (args.gpus, world))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    Bn.load()

    cfg = W.config(args.config)
    B = args.batch or cfg["batch"]
    L = Bn.Landau(cfg["grids"], cfg["species"], cfg["degree"], device=local)
    Bn.landau_set_inner_kernel(L.ctx, args.kernel)
    if args.assembly:
        Bn.landau_set_assembly_kernel(L.ctx, args.assembly)
    if args.chunk:
        Bn.landau_set_batch_chunk(L.ctx, args.chunk)
    coords = [L.dof_coords(g) for g in range(L.G)]
    # weak scaling: rank r owns the global batch entries [r*B, (r+1)*B) -- independent problems, no collective
    entries = sharding.shard_entries(rank, world, B * world, mode="weak")
    f_host = torch.from_numpy(W.make_batch_f(cfg, coords, batch=B * world, entries=entries)).pin_memory()
    out_host = torch.empty((B, L.csr_stride), dtype=torch.float64).pin_memory()
    f_dev = [f_host.to(dev), f_host.to(dev).clone()]  # two input copies, alternated
    out_dev = torch.empty((B, L.csr_stride), dtype=torch.float64, device=dev)
    stream = torch.cuda.current_stream()
    N = int(sum(L.n_ip))
    pairs = float(N) * float(N)

    # FP64 pipe peaks measured in-process (roofline denominator): plain DFMA and DMMA m8n8k4
    peak_dfma = Bn.landau_fp64_probe(0, 20000)
    peak_dmma = Bn.landau_fp64_probe(1, 20000)
    peak = max(peak_dfma, peak_dmma)

    def step(i):
        Bn.landau_jacobian(L.ctx, f_dev[i & 1], B, cfg["dt"], out_dev)

    for i in range(args.warmup):
        step(i)
    Bn.landau_set_timing(L.ctx, 1)
    sampler = ClockSampler(local) if rank == 0 else None
    sharding.barrier(world)
    torch.cuda.synchronize()
    launches0 = Bn.landau_launch_count(L.ctx)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_wall0 = time.perf_counter()
    e0.record(stream)
    stage = np.zeros(4)
    for i in range(args.steps):
        step(i)
        if i == args.steps - 1:
            e1.record(stream)
        stage += np.array(Bn.landau_last_stage_ms(L.ctx))  # waits for this step's last event (host only)
    torch.cuda.synchronize()
    sharding.barrier(world)
    t_wall1 = time.perf_counter()
    ms_total = sharding.max_over_ranks(e0.elapsed_time(e1), world, dev)
    launches = Bn.landau_launch_count(L.ctx) - launches0
    Bn.landau_set_timing(L.ctx, 0)
    clocks = None
    if sampler is not None:
        sampler.stop()
        clocks = sampler.summary(t_wall0, t_wall1)
    ms_per_step = ms_total / args.steps
    value = world * B / (ms_per_step * 1e-3)

    # sanity on the result of the timed steps: finite, and 1^T J = 0 cannot be checked with the shift, so
    # check the mass identity instead: sum of all entries of M/dt - J block = (1/dt) 1^T M 1 (since 1^T J = 0)
    blk = out_dev[0, :int(L.nnz[L.sgrid[0]])]
    g0 = cfg["grids"][L.sgrid[0]]
    expect = g0["r_max"] ** 2 * (g0["z_max"] - g0["z_min"]) / 2.0 / cfg["dt"]
    got = float(blk.sum())
    if not (math.isfinite(got) and abs(got - expect) < 1e-8 * abs(expect)):
        raise SystemExit("bench sanity failed: sum(M/dt - J) = %r, expected %r" % (got, expect))

    # end to end through the C ABI with HOST buffers (H2D of f and D2H of the CSR values inside the timed region)
    e2e = None
    if not args.no_e2e:
        for i in range(2):
            Bn.landau_jacobian_host(L.ctx, f_host, B, cfg["dt"], out_host)
        sharding.barrier(world)
        torch.cuda.synchronize()
        n_e2e = max(2, min(args.steps, 5))
        t0 = time.perf_counter()
        for i in range(n_e2e):
            Bn.landau_jacobian_host(L.ctx, f_host, B, cfg["dt"], out_host)  # synchronous
        torch.cuda.synchronize()
        t_e2e = sharding.max_over_ranks((time.perf_counter() - t0) * 1e3, world, dev) / n_e2e
        # same values up to summation order: the host path runs the batch in pieces, and the persistent K2 cuts the
        # source range of a few tiles at piece-dependent places (K2 stream mode)
        if (args.steps - 1) & 1 == 0:
            a, b = out_host[0].numpy(), out_dev[0].cpu().numpy()
            if not np.linalg.norm(a - b) <= 1e-13 * np.linalg.norm(b):
                raise SystemExit("bench sanity failed: host-buffer path differs from device path")
        e2e = {"value": world * B / (t_e2e * 1e-3), "unit": UNIT, "ms_per_step": t_e2e,
               "h2d_bytes_per_step": int(f_host.numel() * 8), "d2h_bytes_per_step": int(out_host.numel() * 8),
               "steps": n_e2e, "api": "landau_jacobian_host (pinned host buffers)"}

    solve = None
    if args.solve:
        # the step after the hot path: backward-Euler systems (M/dt - J) x = (M/dt) f, TFQMR + Jacobi
        a_inf = torch.empty_like(out_dev)
        Bn.landau_jacobian(L.ctx, f_dev[0], B, float("inf"), a_inf)
        Bn.landau_jacobian(L.ctx, f_dev[0], B, cfg["dt"], out_dev)
        rhs = torch.empty_like(f_dev[0])
        Bn.landau_spmv(L.ctx, out_dev - a_inf, f_dev[0], B, rhs)
        del a_inf
        x = torch.zeros_like(rhs)
        iters = torch.zeros((B, L.S), dtype=torch.int32, device=dev)
        t_solve = []
        for rep in range(3):
            x.zero_()
            s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            s0.record(stream)
            Bn.landau_solve(L.ctx, out_dev, rhs, B, 1e-8, 2000, x, iters)
            s1.record(stream)
            torch.cuda.synchronize()
            t_solve.append(s0.elapsed_time(s1))
        res = rhs - L.spmv(out_dev, x)
        solve = {"ms_per_batch": min(t_solve), "systems": int(B * L.S), "rtol": 1e-8,
                 "half_steps_mean": float(iters.float().abs().mean()), "half_steps_max": int(iters.abs().max()),
                 "not_converged": int((iters < 0).sum()),
                 "max_true_relative_residual": float((res.norm(dim=1) / rhs.norm(dim=1)).max()),
                 "solves_per_s": world * B * L.S / (min(t_solve) * 1e-3)}
    advance = None
    if args.advance:
        # the implicit advance the path belongs to (Table 5): backward-Euler steps of the whole batch
        u = f_dev[0].clone()
        Bn.landau_step(L.ctx, u, B, cfg["dt"], 1e-8, 50, 1e-10, 2000)          # warm-up (scratch, mass values)
        u.copy_(f_dev[0])
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        newton = 0
        for k in range(args.advance):
            info = Bn.landau_step(L.ctx, u, B, cfg["dt"], 1e-8, 50, 1e-10, 2000)
            newton += info["newton_its"]
        torch.cuda.synchronize()
        t_adv = time.perf_counter() - t0
        advance = {"steps": args.advance, "dt": cfg["dt"], "seconds": t_adv, "newton_iterations": newton,
                   "newton_rtol": 1e-8, "lin_rtol": 1e-10, "last": info,
                   "newton_iterations_x_batch_per_s": newton * B * world / t_adv}
    if rank == 0:
        # roofline of the dominant kernel (K2, inner integral).  Algorithmic FLOPs per step:
        # 14 flop per (i, j, source column) -- separable nu: one column per batch entry over all N^2 pairs --
        # plus ONE tensor evaluation per pair (the tensor does not depend on the batch entry).
        cols_pairs = 0.0
        sizes = [int(x) for x in L.n_ip]
        sp_per_grid = [sum(1 for s in L.sgrid if s == g) for g in range(L.G)]
        separable = Bn.landau_is_separable(L.ctx)
        if separable:
            cols_pairs = pairs * B
        else:
            cols_pairs = float(N) * sum(sizes[g] * sp_per_grid[g] for g in range(L.G)) * B
        flop_u = TENSOR_FLOP_PER_PAIR
        alg_flop = cols_pairs * FLOP_PER_PAIR_COLUMN + pairs * flop_u
        k2_ms = stage[1] / args.steps
        achieved = alg_flop / (k2_ms * 1e-3) / 1e12
        k3_ms = stage[3] / args.steps
        csr_bytes = float(B) * L.csr_stride * 8
        dk_bytes = float(B) * L.dk_stride * 8
        traffic = ncu_traffic(workload_name(cfg, B))
        roofline = {"kernel": "K2 inner integral (k2_inner_*)", "bound": "alu", "achieved": achieved, "peak": peak,
                    "unit": "TFLOP/s", "frac": achieved / peak, "traffic": traffic.get("k2_dram_bytes_per_launch"),
                    "traffic_source": traffic.get("source"),
                    "peak_source": "in-process FP64 probe (DFMA %.2f, DMMA m8n8k4 %.2f TFLOP/s), max taken"
                                   % (peak_dfma, peak_dmma),
                    "k2_ms_per_step": k2_ms, "share_of_step": k2_ms / (sum(stage) / args.steps),
                    "algorithmic_flop_per_step": alg_flop,
                    "assembly": {"kernel": "K3 element matrices + assembly (k3_*)", "bound": "hbm",
                                 "achieved": (csr_bytes + dk_bytes) / (k3_ms * 1e-3) / 1e9, "peak": hbm_peak(),
                                 "unit": "GB/s", "frac": (csr_bytes + dk_bytes) / (k3_ms * 1e-3) / 1e9 / hbm_peak(),
                                 "k3_ms_per_step": k3_ms, "algorithmic_bytes_per_step": csr_bytes + dk_bytes,
                                 "traffic": traffic.get("k3_dram_bytes_per_launch")}}
        cpu = None
        if not args.no_cpu_baseline and world == 1:
            v, n_done, threads, times = oracle_sample(cfg, args.cpu_seconds)
            cpu = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle",
                   "sample": "%d Jacobian(s) (batch entries 0..%d) of the workload, %.1f s" % (n_done, n_done - 1, sum(times))}
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": workload_name(cfg, B), "species": L.S, "grids": L.G, "n_ip": N,
                           "pairs_per_jacobian": pairs, "csr_bytes_per_jacobian": int(L.csr_stride * 8),
                           "parallelism": "batch shards, no collective (dp%d)" % world,
                           "l2": "working set per step (CSR out %.2f GB + scratch) exceeds the 126 MB L2; "
                                 "two input copies alternated" % (csr_bytes / 1e9)},
                "pair_evals_per_s": {"tensor_evaluations_unique": pairs * world / (ms_per_step * 1e-3),
                                     # the many-column kernel re-evaluates the tensor once per tile of 256 columns
                                     "tensor_evaluations_executed": pairs * math.ceil(cols_pairs / pairs / 256.0) * world
                                     / (ms_per_step * 1e-3) if separable and cols_pairs / pairs > 128 else None,
                                     "pair_applications_b_i_j": cols_pairs * world / (ms_per_step * 1e-3)},
                "stage_ms_per_step": {"a1_fields": stage[0] / args.steps, "a2_inner": k2_ms,
                                      "a2b_combine": stage[2] / args.steps, "a3a4_assembly": k3_ms},
                "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "solve": solve, "advance": advance, "gpu_launches": int(launches),
                "clocks": clocks}
        print(json.dumps(line), flush=True)
    L.close()
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


def ncu_traffic(workload):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full` capture of this
    workload (profiles/r1_traffic.json.txt); empty when the workload is another one (traffic = null)."""
    try:
        with open(os.path.join(ROOT, "profiles", "r1_traffic.json.txt")) as fh:
            t = json.load(fh)
        return t if workload.startswith(t["workload"]) else {}
    except (OSError, KeyError, ValueError):
        return {}


def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as fh:
            return float(json.load(fh)["hbm_gbs"])
    except (OSError, KeyError, ValueError):
        return 6650.0  # B200_PROFILING.md fallback


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
