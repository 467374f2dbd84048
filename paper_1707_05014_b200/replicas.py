"""Host logic of the N > 1 launch (replicas only).

DROP blocks are sequential in the image, so one solve does not shard; `bench.py --gpus N` runs N
independent replicas, one process per GPU, each on its own slice of the seeded history stream.  There
is no data-path collective: the process group carries the barrier around the timed region and the
max-over-ranks of the device time.  Backend-agnostic (nccl on the GPUs, gloo in the CPU tests).
"""
import torch
import torch.distributed as dist


def shard_first(rank, n_per_rank):
    """First history of rank `rank`'s replica: ranks draw disjoint, contiguous ranges
    [rank * n, (rank + 1) * n) of the same seeded stream."""
    if rank < 0 or n_per_rank <= 0:
        raise ValueError("rank >= 0 and n_per_rank > 0 required")
    return int(rank) * int(n_per_rank)


def barrier(world):
    if world > 1:
        dist.barrier()


def max_over_ranks(value, world, device="cpu"):
    """Max over ranks of a per-rank scalar (the device time of the timed region)."""
    if world == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(ms_local, n_per_rank, steps, world, device="cpu"):
    """(ms of the slowest rank, histories * steps of ALL ranks per second of that time)."""
    ms = max_over_ranks(ms_local, world, device)
    return ms, world * int(n_per_rank) * int(steps) / (ms * 1e-3)
