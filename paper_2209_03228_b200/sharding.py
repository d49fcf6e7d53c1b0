"""Multi-GPU plumbing: batch entries are independent velocity-space problems (PAPER.md:109, 127, 285 -- the paper runs
one MPI rank per GPU, each with its own batch, no communication), so the path shards over the batch with NO
data-path collective.  What is here: which global entries a rank owns, and the two control-plane reductions the
bench needs (barrier, max over ranks of a device-measured time).  Works with the `nccl` backend on GPUs and with
`gloo` on CPU (tests/test_sharding_gloo.py)."""
import os


def env_rank():
    """(rank, world_size, local_rank) from the torchrun environment; (0, 1, 0) outside it."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def shard_entries(rank, world, total, mode="weak"):
    """Global batch-entry ids owned by `rank` out of `total` entries.

    Contiguous ranges; with total not divisible by world the first (total % world) ranks get one entry more
    ("strong" scaling of a fixed batch); mode "weak" requires divisibility (every rank the same work)."""
    if not (0 <= rank < world) or total < 0:
        raise ValueError("bad rank/world/total")
    base, extra = divmod(total, world)
    if mode == "weak" and extra:
        raise ValueError("weak scaling needs total divisible by world")
    lo = rank * base + min(rank, extra)
    return list(range(lo, lo + base + (1 if rank < extra else 0)))


def barrier(world):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def max_over_ranks(value, world, device=None):
    """max over ranks of a Python float (the device-timed milliseconds of each rank)."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def gather_to_rank0(local, world):
    """Concatenate per-rank CPU tensors [n_r, ...] on rank 0 in rank order (only if a single consumer wants the
    whole batch; not used on the timed path)."""
    if world <= 1:
        return local
    import torch
    import torch.distributed as dist
    objs = [None] * world if dist.get_rank() == 0 else None
    dist.gather_object(local, objs, dst=0)
    return torch.cat(objs) if objs is not None else None
