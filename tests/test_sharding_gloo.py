"""N>1 host logic on CPU: world_size-2 gloo run of the batch sharding + the control-plane reductions bench.py uses.
The data path has no collective (entries are independent), so what is covered is that the
shards tile the global batch, that each rank generates exactly its own entries, and that max-over-ranks works."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2209_03228_b200 import sharding
from paper_2209_03228_b200 import workloads as W


def test_shard_entries_tile_the_batch():
    for total in (0, 1, 7, 64, 1000):
        for world in (1, 2, 3, 8):
            got = []
            for r in range(world):
                got += sharding.shard_entries(r, world, total, mode="strong")
            assert got == list(range(total))
            sizes = [len(sharding.shard_entries(r, world, total, mode="strong")) for r in range(world)]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        sharding.shard_entries(0, 2, 7, mode="weak")
    with pytest.raises(ValueError):
        sharding.shard_entries(2, 2, 8)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        assert sharding.env_rank() == (rank, world, rank)
        cfg = W.tiny_config("uniform", 2, batch=3)
        rng = np.random.default_rng(5)
        coords = [rng.uniform(0, 1, (11, 2)), rng.uniform(0, 1, (7, 2))]  # any dof coordinates: generator only
        mine = sharding.shard_entries(rank, world, 3 * world, mode="weak")
        f = torch.from_numpy(W.make_batch_f(cfg, coords, batch=3 * world, entries=mine))
        sharding.barrier(world)
        m = sharding.max_over_ranks(10.0 + rank, world)
        allf = sharding.gather_to_rank0(f, world)
        if rank == 0:
            ref = torch.from_numpy(W.make_batch_f(cfg, coords, batch=3 * world))
            q.put(("ok", m, bool(torch.equal(allf, ref))))
    finally:
        dist.destroy_process_group()


def test_world2_gloo_shards_and_reductions():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    tag, m, same = q.get(timeout=10)
    assert tag == "ok" and m == 11.0 and same


def test_bench_gpus_n_starts_n_ranks():
    """`python bench.py --gpus 2` outside a torchrun environment must really run two ranks (here: --dry-run, gloo, no GPU work)
    and say so in its line -- it used to benchmark one GPU silently."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--dry-run", "--config", "2", "--batch", "8"],
                         capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                                   # rank 0 alone prints
    line = json.loads(lines[0])
    assert line["n_gpus"] == 2 and line["dry_run"] is True
    assert line["shards"] == [[0, 0, 7], [1, 8, 15]]          # weak scaling: rank r owns entries [8 r, 8 r + 8)
    assert line["max_over_ranks_ms"] == 2.0                   # max over ranks of (1 + rank)
