"""Multi-GPU plumbing for bench.py: one process per GPU, N independent replicas of the path.

The MD step of one lattice does not shard without a halo exchange (not built),
so N > 1 runs N independent lattices -- "replicas only", weak scaling, no data-path collective.
torch.distributed is used for the barrier around the timed region and for two tiny reductions:
the MAX over ranks of the device time and the SUM over ranks of the work done.
"""
import os


def env_rank_world():
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def init(backend, device=None):
    """Initialises the default process group from the torchrun environment (no-op for world size 1)."""
    import torch.distributed as dist

    rank, world, _ = env_rank_world()
    if world > 1 and not dist.is_initialized():
        kw = {"device_id": device} if device is not None else {}
        dist.init_process_group(backend, **kw)
    return rank, world


def barrier():
    import torch.distributed as dist

    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def aggregate(times, sums, device="cpu"):
    """times: per-rank durations -> elementwise MAX over ranks; sums: per-rank work counts -> SUM over ranks.
    Returns (times_max, sums_total) as python lists; identity for a single process."""
    import torch
    import torch.distributed as dist

    t = torch.tensor(list(times), dtype=torch.float64, device=device)
    s = torch.tensor(list(sums), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized():
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(s, op=dist.ReduceOp.SUM)
    return t.tolist(), s.tolist()


def throughput(units_total, time_max_s):
    """Whole-job throughput: units all ranks processed / max-over-ranks time."""
    return units_total / time_max_s


def shutdown():
    import torch.distributed as dist

    if dist.is_available() and dist.is_initialized():
        dist.destroy_process_group()
