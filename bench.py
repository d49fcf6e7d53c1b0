#!/usr/bin/env python
"""bench.py -- throughput of the batched Landau Jacobian construction (BASELINE.json metric) on N B200s.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 5] [--batch 1024] [--impl ours|reference]

One "step" = one pass of the whole hot path (a1 field evaluation, a2 inner integral, a2b species combination,
a3+a4 element matrices + assembly into the batched CSR of M/dt - J) over one batch of seeded synthetic
distribution functions.  Default workload: BASELINE.json configs[4] ("large-batch
throughput ... Jacobian build + assembly timed end to end"), e-/D+ on uniform 14x28 Q3 grids, batch 1024 per GPU
(DESIGN.md "Measurement" says why this one and not configs[1]; `--config 2 --batch 64` runs configs[1]).
`--config 6` is the paper's own 2V throughput problem, `--config 7` the paper's 3V problem (ten species, three grids of
120 Q2 hexahedra, batch 32; Table 6), `--config 8` e-/D+ on two such 3V grids.

Prints ONE JSON line (rank 0): value = Landau Jacobians/s of the whole job, device-resident inputs; e2e = same
metric through landau_jacobian_host (pinned HOST buffers, H2D + D2H inside the timed region); roofline = the
inner-integral kernel (K2) against the FP64 pipe peak measured in-process (nominal figure beside it), with the assembly
kernel (K3) against the measured HBM bandwidth under "assembly"; cpu_baseline = the oracle, as it stands, on the host
cores over a bounded sample of the same workload.  Extras that do not enter `value`:
  other_configs  short runs (3 steps) of the other BASELINE.json configs and of the paper's 3V problem: Jacobians/s, stage
                 times, K2 and K3 roofline fractions (skip with --no-other-configs)
  solve          the batched TFQMR + Jacobi solve of the step's backward-Euler systems on a bounded sub-batch
                 (148 entries; the whole batch with --solve)
  advance        three backward-Euler steps (landau_step) of the paper's 2V throughput problem, Newton iterations x batch per
                 second; `--advance N`: N steps of the headline workload instead

`--gpus N` without a torchrun environment starts N ranks itself (one per GPU; NCCL for the barrier and the max-reduce
only: batch entries are independent); `--dry-run` exercises that plumbing without a GPU (gloo).
`--impl reference` times the oracle only (no GPU work); under torchrun only rank 0 runs it.
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
# Algorithmic FP64 work of the inner integral: FMAs x 2 per (i, j, source column), plus ONE
# tensor evaluation per pair.  The cost of an evaluation comes from the ncu instruction totals of the committed capture
# (profiles/r2_traffic.json.txt: thread-level dfma / dmul / dadd counts of K2 divided by the evaluations it executed);
# the constants below are only the fall-back when that file does not cover the kernel.
FLOP_PER_PAIR_COLUMN = {2: 14.0, 3: 30.0}
TENSOR_FLOP_FALLBACK = {2: 140.0, 3: 40.0}
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12   # 148 SMs x 64 FMA/clk x 2 x 1.965 GHz (guide: unit counts, max clock)


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5, help="BASELINE.json config number 1..5 (6: the paper's 2V throughput "
                    "problem, 7: the paper's 3V problem, 8: e-/D+ in 3V)")
    ap.add_argument("--batch", type=int, default=None, help="batch entries PER GPU (default: the config's)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="CPU time budget of the cpu_baseline sample")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true", help="skip the short runs of the other configs")
    ap.add_argument("--no-solve", action="store_true", help="skip the bounded TFQMR solve")
    ap.add_argument("--kernel", type=int, default=0, help="inner-integral kernel: 0 auto, 1 DFMA, 2 DMMA, 3/4/5 GEMM (16x128 / 16x256 / 16x64 tile)")
    ap.add_argument("--solve", action="store_true", help="time the batched TFQMR solve on the WHOLE batch (default: 148 entries)")
    ap.add_argument("--advance", type=int, default=0, help="also run this many backward-Euler steps (landau_step) and "
                    "report the time and Newton iterations under \"advance\" (not part of value)")
    ap.add_argument("--assembly", type=int, default=0, help="assembly kernel build (landau_set_assembly_kernel; 0: default)")
    ap.add_argument("--chunk", type=int, default=0, help="batch entries per pass through the stages (0: library default)")
    ap.add_argument("--print-csrc-hash", action="store_true", help="print the sha256 that identifies the kernel sources and exit")
    ap.add_argument("--dry-run", action="store_true", help="rank plumbing only (gloo, no GPU work): the CPU test of --gpus N")
    return ap.parse_args()


def load_config(index, batch=None):
    """(cfg, dim): BASELINE.json configs 1..5, the paper's 2V problem (6) and the 3V problems (7, 8)."""
    from paper_2209_03228_b200 import workloads as W
    if index in (7, 8):
        return W.config3v("paper" if index == 7 else "eD", batch), 3
    return W.config(index, batch), 2


def workload_name(cfg, B):
    if cfg["index"] <= 5:
        return "%s batch=%d/GPU (BASELINE.json configs[%d])" % (cfg["name"], B, cfg["index"] - 1)
    return "%s batch=%d/GPU (the paper's own problem, PAPER.md:125)" % (cfg["name"], B)


TRAFFIC_FILE = os.path.join("profiles", "r3_traffic.json.txt")


def csrc_sha256():
    """sha256 over the CUDA / C++ sources of the library (file names and contents, sorted by name): the build the ncu
    counters in TRAFFIC_FILE were captured on is identified by it (`python bench.py --print-csrc-hash`)."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2209_03228_b200", "csrc")
    for name in sorted(os.listdir(d)):
        if name.endswith((".cu", ".cuh", ".cpp", ".hpp", ".h")):
            h.update(name.encode())
            with open(os.path.join(d, name), "rb") as fh:
                h.update(fh.read())
    return h.hexdigest()


def profile_data():
    """Per-launch ncu figures of the committed `ncu --set full` captures (TRAFFIC_FILE).  They describe ONE build: when the
    sources have changed since the capture, nothing from the file is used (traffic: null, tensor FLOP: fall-back constant)
    instead of carrying stale counters."""
    try:
        with open(os.path.join(ROOT, TRAFFIC_FILE)) as fh:
            prof = json.load(fh)
    except (OSError, ValueError):
        return {"source": None}
    if prof.get("csrc_sha256") != csrc_sha256():
        return {"source": "%s is stale: captured on csrc sha256 %s" % (TRAFFIC_FILE, str(prof.get("csrc_sha256"))[:16])}
    return prof


def hbm_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return float(json.load(fh)["hbm_gbs"]), "MEASURED_PEAKS.json"
    except (OSError, KeyError, ValueError):
        return 6650.0, "fallback (B200_PROFILING.md)"


class Problem:
    """One context (2V: binding.Landau, 3V: binding3v.Landau3V) behind the calls the measurement needs."""

    def __init__(self, cfg, dim, device, kernel=0, assembly=0, chunk=0):
        from paper_2209_03228_b200 import workloads as W
        self.cfg, self.dim = cfg, dim
        if dim == 2:
            from paper_2209_03228_b200 import binding as Bn
            self.Bn = Bn
            self.L = Bn.Landau(cfg["grids"], cfg["species"], cfg["degree"], device=device)
            Bn.landau_set_inner_kernel(self.L.ctx, kernel)
            if assembly:
                Bn.landau_set_assembly_kernel(self.L.ctx, assembly)
            if chunk:
                Bn.landau_set_batch_chunk(self.L.ctx, chunk)
            self.separable = bool(Bn.landau_is_separable(self.L.ctx))
            self.make_f = W.make_batch_f
        else:
            from paper_2209_03228_b200 import binding3v as B3
            self.Bn = B3
            self.L = B3.Landau3V(cfg["grids"], cfg["species"], device=device)
            if kernel:
                B3.landau3v_set_inner_kernel(self.L.ctx, min(kernel, 3))
            if assembly:
                B3.landau3v_set_assembly_kernel(self.L.ctx, 1 if assembly == 1 else 0)
            if chunk:
                B3.landau3v_set_batch_chunk(self.L.ctx, chunk)
            self.separable = True   # nu = q_a^2 q_b^2 is rank one
            self.make_f = W.make_batch_f3v
        self.N = int(sum(self.L.n_ip))
        self.csr_stride, self.dk_stride, self.f_stride = int(self.L.csr_stride), int(self.L.dk_stride), int(self.L.f_stride)

    def coords(self):
        return [self.L.dof_coords(g) for g in range(self.L.G)]

    def jacobian(self, f, B, out):
        (self.Bn.landau_jacobian if self.dim == 2 else self.Bn.landau3v_jacobian)(self.L.ctx, f, B, self.cfg["dt"], out)

    def jacobian_host(self, f_host, B, out_host):
        (self.Bn.landau_jacobian_host if self.dim == 2 else self.Bn.landau3v_jacobian_host)(
            self.L.ctx, f_host, B, self.cfg["dt"], out_host)

    def set_timing(self, on):
        (self.Bn.landau_set_timing if self.dim == 2 else self.Bn.landau3v_set_timing)(self.L.ctx, 1 if on else 0)

    def stage_ms(self):
        return np.array((self.Bn.landau_last_stage_ms if self.dim == 2 else self.Bn.landau3v_last_stage_ms)(self.L.ctx))

    def launches(self):
        return (self.Bn.landau_launch_count if self.dim == 2 else self.Bn.landau3v_launch_count)(self.L.ctx)

    def pair_work(self, B):
        """(unique tensor pairs, (i, j, column) products) of one step of B entries."""
        pairs = float(self.N) * float(self.N)
        if self.separable:
            return pairs, pairs * B
        sizes = [int(x) for x in self.L.n_ip]
        per_grid = [sum(1 for s in self.L.sgrid if s == g) for g in range(self.L.G)]
        return pairs, float(self.N) * sum(sizes[g] * per_grid[g] for g in range(self.L.G)) * B

    def mass_block_sum(self):
        """sum of all entries of the first species' block of M/dt - J = (1/dt) 1^T M 1 (since 1^T J = 0): the grid's measure."""
        g0 = self.cfg["grids"][self.L.sgrid[0]]
        vol = (2 * g0["half"]) ** 3 if self.dim == 3 else g0["r_max"] ** 2 * (g0["z_max"] - g0["z_min"]) / 2.0
        return vol / self.cfg["dt"], int(self.L.nnz[self.L.sgrid[0]])

    def close(self):
        self.L.close()


# ----------------------------------------------------------------------------------------------------------------
# the oracle arm: cpu_baseline leg and --impl reference
# ----------------------------------------------------------------------------------------------------------------
def open_oracle(cfg, dim):
    """(oracle object, make_batch_f) for a 2V or a 3V problem."""
    from paper_2209_03228_b200 import workloads as W
    if dim == 3:
        from oracle import oracle3v as O3
        O3.build()
        return O3.Oracle3V(cfg["grids"], cfg["species"]), W.make_batch_f3v
    from oracle import oracle as O
    O.build()
    return O.Oracle(cfg["grids"], cfg["species"], cfg["degree"]), W.make_batch_f


def oracle_sample(cfg, dim, seconds, min_entries=1, max_entries=64):
    """Time the oracle (as it stands, OpenMP over field points) on entries 0, 1, ... of the workload until
    `seconds` of wall time are used.  Returns (Jacobians/s, entries done, threads, per-entry seconds)."""
    o, make_f = open_oracle(cfg, dim)
    coords = [o.dof_coords(g) for g in range(o.G)]
    times = []
    t_start = time.perf_counter()
    b = 0
    while b < max_entries and (b < min_entries or time.perf_counter() - t_start < seconds):
        f = make_f(cfg, coords, entries=[b])[0]
        t0 = time.perf_counter()
        o.jacobian(f, cfg["dt"])
        times.append(time.perf_counter() - t0)
        b += 1
    return len(times) / sum(times), len(times), o.threads, times


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg, dim = load_config(args.config)
    B = args.batch or cfg["batch"]
    # a step = a bounded sample: ONE Jacobian (entry s mod B) of the workload on all host cores
    o, make_f = open_oracle(cfg, dim)
    coords = [o.dof_coords(g) for g in range(o.G)]
    fs = [make_f(cfg, coords, entries=[s % B])[0] for s in range(args.steps + args.warmup)]
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
def tensor_flop(dim, prof):
    """FP64 FLOP of one tensor evaluation: ncu thread-instruction totals of K2 (2 x dfma + dmul + dadd; the DMMA
    accumulation is a separate op class) divided by the evaluations the captured launch executed."""
    key = "k2" if dim == 2 else "k2_3v"
    try:
        ev = float(prof[key + "_tensor_evaluations_executed"])
        return (2.0 * prof[key + "_thread_inst_dfma"] + prof[key + "_thread_inst_dmul"] + prof[key + "_thread_inst_dadd"]) / ev, \
            "ncu (%s)" % TRAFFIC_FILE
    except (KeyError, TypeError, ZeroDivisionError):
        return TENSOR_FLOP_FALLBACK[dim], "fall-back"


def rooflines(P, B, stage_ms, fp64_peak, prof, workload):
    """Roofline objects of K2 (inner integral, FP64 pipe) and K3 (assembly, HBM) from the stage times of one step."""
    pairs, cols_pairs = P.pair_work(B)
    flop_u, flop_src = tensor_flop(P.dim, prof)
    alg_flop = cols_pairs * FLOP_PER_PAIR_COLUMN[P.dim] + pairs * flop_u
    k2_ms, k3_ms = float(stage_ms[1]), float(stage_ms[3])
    achieved = alg_flop / (k2_ms * 1e-3) / 1e12
    hbm, hbm_src = hbm_peak()
    alg_bytes = float(B) * (P.csr_stride + P.dk_stride) * 8
    tag = "" if P.dim == 2 else "_3v"
    same = str(prof.get("workload" + tag, "")) and workload.startswith(str(prof.get("workload" + tag, "")))
    k2 = {"kernel": "K2 inner integral (%s)" % ("k2_inner_*" if P.dim == 2 else "k3v_inner_*"), "bound": "alu",
          "achieved": achieved, "peak": fp64_peak, "unit": "TFLOP/s", "frac": achieved / fp64_peak,
          "traffic": prof.get("k2%s_dram_bytes_per_launch" % tag) if same else None,
          "k2_ms_per_step": k2_ms, "share_of_step": k2_ms / float(sum(stage_ms)), "algorithmic_flop_per_step": alg_flop,
          "tensor_flop_per_evaluation": flop_u, "tensor_flop_source": flop_src}
    k3 = {"kernel": "K3 element matrices + assembly (%s)" % ("k3_ring" if P.dim == 2 else "k3v_elem_matrix + k3v_gather"),
          "bound": "hbm", "achieved": alg_bytes / (k3_ms * 1e-3) / 1e9, "peak": hbm, "peak_source": hbm_src, "unit": "GB/s",
          "frac": alg_bytes / (k3_ms * 1e-3) / 1e9 / hbm, "k3_ms_per_step": k3_ms, "algorithmic_bytes_per_step": alg_bytes,
          "traffic": prof.get("k3%s_dram_bytes_per_launch" % tag) if same else None}
    return k2, k3


def measure(P, B, steps, warmup, f_dev, out_dev, world, dev, sharding, sampler_index=None):
    """`warmup` untimed + `steps` timed steps (CUDA events on the launching stream, barrier + synchronize on both sides, max
    over ranks).  Returns (ms per step, stage ms per step, launches in the timed region, clocks summary or None)."""
    import torch
    stream = torch.cuda.current_stream()
    for i in range(warmup):
        P.jacobian(f_dev[i & 1], B, out_dev)
    P.set_timing(True)
    sampler = ClockSampler(sampler_index) if sampler_index is not None else None
    sharding.barrier(world)
    torch.cuda.synchronize()
    launches0 = P.launches()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_wall0 = time.perf_counter()
    e0.record(stream)
    stage = np.zeros(4)
    for i in range(steps):
        P.jacobian(f_dev[i & 1], B, out_dev)
        if i == steps - 1:
            e1.record(stream)
        stage += P.stage_ms()  # waits for this step's last event (host only)
    torch.cuda.synchronize()
    sharding.barrier(world)
    t_wall1 = time.perf_counter()
    ms_total = sharding.max_over_ranks(e0.elapsed_time(e1), world, dev)
    launches = P.launches() - launches0
    P.set_timing(False)
    clocks = None
    if sampler is not None:
        sampler.stop()
        clocks = sampler.summary(t_wall0, t_wall1)
    return ms_total / steps, stage / steps, int(launches), clocks


def sanity(P, out_dev):
    expect, n0 = P.mass_block_sum()
    got = float(out_dev[0, :n0].sum())
    if not (math.isfinite(got) and abs(got - expect) < 1e-8 * abs(expect)):
        raise SystemExit("bench sanity failed: sum(M/dt - J) = %r, expected %r" % (got, expect))


def other_config_runs(local, dev, fp64_peak, prof, skip):
    """Short runs of the configs BASELINE.json lists besides the headline one, and of the paper's 3V problem."""
    import torch
    from paper_2209_03228_b200 import sharding
    rows = []
    plan = [(1, 1), (2, 64), (3, 1), (3, 16), (3, 64), (3, 256), (3, 512), (4, 256), (5, 1024), (5, 4096), (7, 32)]
    probs = {}
    for index, B in plan:
        if (index, B) == skip:
            continue
        try:
            if index not in probs:
                for P in probs.values():
                    P.close()
                probs = {}
                cfg, dim = load_config(index)
                probs[index] = Problem(cfg, dim, local)
            P = probs[index]
            f = torch.from_numpy(P.make_f(P.cfg, P.coords(), batch=B)).to(dev)
            out = torch.empty((B, P.csr_stride), dtype=torch.float64, device=dev)
            ms, stage, launches, _ = measure(P, B, 3, 2, [f, f], out, 1, dev, sharding)
            sanity(P, out)
            if ms < 10.0:
                # short steps: the stage timing above waits for every step on the host, which leaves the launch latency of a
                # step exposed; time about 30 ms of steps issued back to back for the throughput figure
                n = int(min(200, max(3, 30.0 / ms)))
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize()
                e0.record()
                for _ in range(n):
                    P.jacobian(f, B, out)
                e1.record()
                torch.cuda.synchronize()
                ms = e0.elapsed_time(e1) / n
            k2, k3 = rooflines(P, B, stage, fp64_peak, prof, "")
            rows.append({"workload": workload_name(P.cfg, B), "jacobians_per_s": B / (ms * 1e-3), "ms_per_step": ms,
                         "stage_ms": {"a1": stage[0], "a2": stage[1], "a2b": stage[2], "a3a4": stage[3]},
                         "k2_tflops": k2["achieved"], "k2_frac": k2["frac"], "k3_gbs": k3["achieved"], "k3_frac": k3["frac"],
                         "launches_per_step": launches / 3})
            del f, out
        except Exception as e:  # a failing extra must not take the headline number with it
            rows.append({"workload": "config %d batch %d" % (index, B), "error": repr(e)[:200]})
    for P in probs.values():
        P.close()
    torch.cuda.empty_cache()
    return rows


def advance_run(local, dev, steps=3, config=6):
    """The implicit advance the path belongs to, bounded: `steps` backward-Euler steps (landau_step / landau3v_step:
    quasi-Newton on the sparse Jacobian, batched TFQMR) of the paper's own throughput problems -- config 6: 2V, ten species,
    three grids of 14 Q3 cells, batch 256; config 7: 3V, three grids of 120 Q2 cells, batch 32 (Tables 5-6).
    Newton iterations x batch per second is the paper's throughput measure."""
    import torch
    cfg, dim = load_config(config)
    B = cfg["batch"]
    P = Problem(cfg, dim, local)
    step = P.Bn.landau_step if dim == 2 else P.Bn.landau3v_step
    f = torch.from_numpy(P.make_f(cfg, P.coords(), batch=B)).to(dev)
    u = f.clone()
    step(P.L.ctx, u, B, cfg["dt"], 1e-8, 50, 1e-10, 2000)          # warm-up (scratch, mass values)
    u.copy_(f)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    newton, info = 0, None
    for k in range(steps):
        info = step(P.L.ctx, u, B, cfg["dt"], 1e-8, 50, 1e-10, 2000)
        newton += info["newton_its"]
    torch.cuda.synchronize()
    t_adv = time.perf_counter() - t0
    P.close()
    return {"workload": workload_name(cfg, B), "steps": steps, "dt": cfg["dt"], "seconds": t_adv, "newton_iterations": newton,
            "newton_rtol": 1e-8, "lin_rtol": 1e-10, "last": info, "newton_iterations_x_batch_per_s": newton * B / t_adv}


def solve_run(P, B, f_dev0, out_dev, dev, whole):
    """The step after the hot path: backward-Euler systems (M/dt - J) x = (M/dt) f of a bounded
    sub-batch, TFQMR + Jacobi, one system per CTA."""
    import torch
    Bn, L, cfg = P.Bn, P.L, P.cfg
    nb = B if whole else min(B, 148)
    f = f_dev0[:nb].contiguous()
    a = torch.empty((nb, P.csr_stride), dtype=torch.float64, device=dev)
    a_inf = torch.empty_like(a)
    Bn.landau_jacobian(L.ctx, f, nb, float("inf"), a_inf)
    Bn.landau_jacobian(L.ctx, f, nb, cfg["dt"], a)
    rhs = torch.empty_like(f)
    Bn.landau_spmv(L.ctx, a - a_inf, f, nb, rhs)
    del a_inf
    x = torch.zeros_like(rhs)
    iters = torch.zeros((nb, L.S), dtype=torch.int32, device=dev)
    stream = torch.cuda.current_stream()
    t_solve = []
    for rep in range(3):
        x.zero_()
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s0.record(stream)
        Bn.landau_solve(L.ctx, a, rhs, nb, 1e-8, 2000, x, iters)
        s1.record(stream)
        torch.cuda.synchronize()
        t_solve.append(s0.elapsed_time(s1))
    res = rhs - L.spmv(a, x)
    ms = min(t_solve)
    # bytes one half-step of one system moves through the SM (one SpMV: values + column indices, plus ~10 vector passes)
    half = iters.abs().to(torch.float64).cpu().numpy()
    byts = 0.0
    for s in range(L.S):
        g = L.sgrid[s]
        byts += float(half[:, s].sum()) * (12.0 * float(L.nnz[g]) + 10 * 8.0 * float(L.n_dof[g]))
    # Denominator.  Small systems: matrix and vectors live in shared memory for the whole iteration -> all bytes go through
    # the shared-memory crossbar, 128 B/clk per SM (B300_MICROARCH.md, LDS/STS table) x 148 SMs x the SM clock.  Larger
    # systems: vectors in shared memory, the matrix streams from L2 in every product -> matrix bytes against the L2 read
    # bandwidth measured by the in-process probe (the guides state no L2 figure).
    mat_bytes = sum(float(half[:, s].sum()) * 12.0 * float(L.nnz[L.sgrid[s]]) for s in range(L.S))
    if Bn.landau_solve_matrix_in_shared(L.ctx):
        bound, ach = "smem", byts / (ms * 1e-3) / 1e9
        peak = 148 * 128.0 * 1.965e9 / 1e9
        peak_src = "148 SM x 128 B/clk (shared-memory crossbar, B300_MICROARCH.md) x 1.965 GHz"
    else:
        bound, ach = "l2", mat_bytes / (ms * 1e-3) / 1e9
        peak = Bn.landau_l2_probe(32 << 20, 64)
        peak_src = "in-process L2 read probe (landau_l2_probe: 32 MiB buffer, 16-byte ld.global.cg, all SMs)"
    return {"ms_per_batch": ms, "entries": int(nb), "systems": int(nb * L.S), "rtol": 1e-8,
            "half_steps_mean": float(half.mean()), "half_steps_max": int(half.max()),
            "not_converged": int((iters < 0).sum()),
            "max_true_relative_residual": float((res.norm(dim=1) / rhs.norm(dim=1)).max()),
            "solves_per_s": nb * L.S / (ms * 1e-3),
            "roofline": {"kernel": "K4 batched TFQMR (k4_tfqmr)", "bound": bound, "achieved": ach, "unit": "GB/s",
                         "peak": peak, "frac": ach / peak, "peak_source": peak_src,
                         "bytes_model": "per half-step of a system: one product = 12 B x nnz (values + column indices)"
                                        + (" + ~10 vector passes of 8 B x n" if bound == "smem" else
                                           "; the ~10 vector passes per half-step stay in shared memory and are not counted")}}


def run_dry(args):
    """--dry-run: the N-rank plumbing without a GPU (gloo): shards, barrier, max over ranks, one JSON line from rank 0."""
    import torch
    import torch.distributed as dist
    from paper_2209_03228_b200 import sharding
    rank, world, local = sharding.env_rank()
    if world > 1:
        dist.init_process_group("gloo")
    cfg, dim = load_config(args.config)
    B = args.batch or cfg["batch"]
    entries = sharding.shard_entries(rank, world, B * world, mode="weak")
    sharding.barrier(world)
    ms = sharding.max_over_ranks(1.0 + rank, world, torch.device("cpu"))
    counts = [None] * world
    if world > 1:
        dist.all_gather_object(counts, (rank, entries[0], entries[-1]))
    else:
        counts = [(0, entries[0], entries[-1])]
    if rank == 0:
        print(json.dumps({"metric": METRIC, "value": None, "unit": UNIT, "n_gpus": world, "dry_run": True,
                          "max_over_ranks_ms": ms, "shards": counts,
                          "config": {"workload": workload_name(cfg, B), "parallelism": "batch shards, no collective (dp%d)" % world}}),
              flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_ours(args):
    import torch
    from paper_2209_03228_b200 import binding as Bn
    from paper_2209_03228_b200 import sharding

    rank, world, local = sharding.env_rank()
    if world != args.gpus:
        raise SystemExit("--gpus %d but WORLD_SIZE=%d" % (args.gpus, world))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    if local >= torch.cuda.device_count():
        raise SystemExit("rank %d has no GPU (%d visible)" % (rank, torch.cuda.device_count()))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    Bn.load()

    cfg, dim = load_config(args.config)
    B = args.batch or cfg["batch"]
    P = Problem(cfg, dim, local, args.kernel, args.assembly, args.chunk)
    # weak scaling: rank r owns the global batch entries [r*B, (r+1)*B) -- independent problems, no collective
    entries = sharding.shard_entries(rank, world, B * world, mode="weak")
    f_host = torch.from_numpy(P.make_f(cfg, P.coords(), batch=B * world, entries=entries)).pin_memory()
    out_host = torch.empty((B, P.csr_stride), dtype=torch.float64).pin_memory()
    f_dev = [f_host.to(dev), f_host.to(dev).clone()]  # two input copies, alternated
    out_dev = torch.empty((B, P.csr_stride), dtype=torch.float64, device=dev)
    pairs, cols_pairs = P.pair_work(B)

    # FP64 pipe peaks measured in-process (roofline denominator): plain DFMA and DMMA m8n8k4
    peak_dfma = Bn.landau_fp64_probe(0, 20000)
    peak_dmma = Bn.landau_fp64_probe(1, 20000)
    peak = max(peak_dfma, peak_dmma)
    prof = profile_data()

    ms_per_step, stage, launches, clocks = measure(P, B, args.steps, args.warmup, f_dev, out_dev, world, dev, sharding,
                                                   local if rank == 0 else None)
    value = world * B / (ms_per_step * 1e-3)
    per_rank = None
    if world > 1:
        import torch.distributed as dist
        mine = torch.tensor([B / (ms_per_step * 1e-3)], dtype=torch.float64, device=dev)
        allv = [torch.zeros_like(mine) for _ in range(world)]
        dist.all_gather(allv, mine)
        per_rank = [float(v.item()) for v in allv]
    sanity(P, out_dev)

    # end to end through the C ABI with HOST buffers (H2D of f and D2H of the CSR values inside the timed region)
    e2e = None
    if not args.no_e2e:
        for i in range(2):
            P.jacobian_host(f_host, B, out_host)
        sharding.barrier(world)
        torch.cuda.synchronize()
        n_e2e = max(2, min(args.steps, 5))
        t0 = time.perf_counter()
        for i in range(n_e2e):
            P.jacobian_host(f_host, B, out_host)  # synchronous
        torch.cuda.synchronize()
        t_e2e = sharding.max_over_ranks((time.perf_counter() - t0) * 1e3, world, dev) / n_e2e
        # same values up to summation order: the host path runs the batch in pieces, and the persistent K2 cuts the
        # source range of a few tiles at piece-dependent places (K2 stream mode)
        a, b = out_host[0].numpy(), out_dev[0].cpu().numpy()
        if not np.linalg.norm(a - b) <= 1e-13 * np.linalg.norm(b):
            raise SystemExit("bench sanity failed: host-buffer path differs from device path")
        e2e = {"value": world * B / (t_e2e * 1e-3), "unit": UNIT, "ms_per_step": t_e2e,
               "h2d_bytes_per_step": int(f_host.numel() * 8), "d2h_bytes_per_step": int(out_host.numel() * 8),
               "steps": n_e2e, "api": "landau%s_jacobian_host (pinned host buffers)" % ("" if dim == 2 else "3v")}

    solve = None
    if dim == 2 and not args.no_solve and rank == 0:
        solve = solve_run(P, B, f_dev[0], out_dev, dev, args.solve)
    advance = None
    if args.advance and dim == 2:
        # the implicit advance the path belongs to (Table 5): backward-Euler steps of the whole batch
        u = f_dev[0].clone()
        Bn.landau_step(P.L.ctx, u, B, cfg["dt"], 1e-8, 50, 1e-10, 2000)          # warm-up (scratch, mass values)
        u.copy_(f_dev[0])
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        newton = 0
        for k in range(args.advance):
            info = Bn.landau_step(P.L.ctx, u, B, cfg["dt"], 1e-8, 50, 1e-10, 2000)
            newton += info["newton_its"]
        torch.cuda.synchronize()
        t_adv = time.perf_counter() - t0
        advance = {"steps": args.advance, "dt": cfg["dt"], "seconds": t_adv, "newton_iterations": newton,
                   "newton_rtol": 1e-8, "lin_rtol": 1e-10, "last": info,
                   "newton_iterations_x_batch_per_s": newton * B * world / t_adv}
    if rank == 0:
        name = workload_name(cfg, B)
        k2, k3 = rooflines(P, B, stage, peak, prof, name)
        k2.update({"peak_probe": peak, "peak_nominal": FP64_NOMINAL_TFLOPS,
                   "peak_source": "in-process FP64 probe (DFMA %.2f, DMMA m8n8k4 %.2f TFLOP/s), max taken; nominal "
                                  "148 SM x 64 FMA/clk x 2 x 1.965 GHz = %.2f" % (peak_dfma, peak_dmma, FP64_NOMINAL_TFLOPS),
                   "traffic_source": prof.get("source"), "assembly": k3})
        cpu = None
        if not args.no_cpu_baseline and world == 1:
            v, n_done, threads, times = oracle_sample(cfg, dim, args.cpu_seconds)
            cpu = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle",
                   "sample": "%d Jacobian(s) (batch entries 0..%d) of the workload, %.1f s" % (n_done, n_done - 1, sum(times))}
        csr_bytes = float(B) * P.csr_stride * 8
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": name, "species": P.L.S, "grids": P.L.G, "n_ip": P.N,
                           "pairs_per_jacobian": pairs, "csr_bytes_per_jacobian": int(P.csr_stride * 8),
                           "parallelism": "batch shards, no collective (dp%d)" % world,
                           "l2": "working set per step (CSR out %.2f GB + scratch) %s the 126 MB L2; two input copies "
                                 "alternated" % (csr_bytes / 1e9, "exceeds" if csr_bytes > 126e6 else "is below")},
                "pair_evals_per_s": {"tensor_evaluations_unique": pairs * world / (ms_per_step * 1e-3),
                                     # the many-column 2V kernel re-evaluates the tensor once per tile of 256 columns, the 3V
                                     # kernel once per tile of 32
                                     "tensor_evaluations_executed": pairs * math.ceil(cols_pairs / pairs / (256.0 if dim == 2 else 32.0))
                                     * world / (ms_per_step * 1e-3) if P.separable and (dim == 3 or cols_pairs / pairs > 128) else None,
                                     "pair_applications_b_i_j": cols_pairs * world / (ms_per_step * 1e-3)},
                "stage_ms_per_step": {"a1_fields": stage[0], "a2_inner": stage[1], "a2b_combine": stage[2], "a3a4_assembly": stage[3]},
                "roofline": k2, "cpu_baseline": cpu, "e2e": e2e, "solve": solve, "advance": advance,
                "gpu_launches": int(launches), "clocks": clocks}
        if per_rank is not None:
            line["per_rank_jacobians_per_s"] = per_rank
    # the context of the headline run is released before the extras so that config 5 at batch 4096 (5.8 GB of CSR) fits
    del f_dev, out_dev
    P.close()
    torch.cuda.empty_cache()
    if rank == 0:
        if not args.no_other_configs and world == 1:
            line["other_configs"] = other_config_runs(local, dev, peak, prof, (args.config, B))
            if line["advance"] is None:
                try:
                    line["advance"] = advance_run(local, dev)
                    line["advance_3v"] = advance_run(local, dev, config=7)
                except Exception as e:  # an extra must not take the headline number with it
                    line["advance" if line["advance"] is None else "advance_3v"] = {"error": repr(e)[:200]}
        print(json.dumps(line), flush=True)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


def spawn_ranks(args):
    """`--gpus N` outside a torchrun environment: start N ranks of this script (one per GPU) the way the driver would and
    pass their output through.  Rank 0 prints the JSON line."""
    import socket
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


if __name__ == "__main__":
    a = parse()
    if a.print_csrc_hash:
        print(csrc_sha256())
        sys.exit(0)
    if a.gpus > 1 and "WORLD_SIZE" not in os.environ:
        spawn_ranks(a)
    if a.impl == "reference":
        run_reference(a)
    elif a.dry_run:
        run_dry(a)
    else:
        run_ours(a)
