"""Host logic of the N > 1 launch.

DROP blocks are sequential in the image, so one DROP solve does not shard; `bench.py --gpus N` runs N
independent replicas, one process per GPU, each on its own slice of the seeded history stream.  There
is no data-path collective there: the process group carries the barrier around the timed region and
the max-over-ranks of the device time.

CARP does shard ("CARP is highly suitable for parallel implementation"): one string per
rank, and the one exchange step of the method -- "a new solution is then computed from the average of
the different string solutions" -- is an all-reduce of the image per iteration (`carp_distributed`).

Backend-agnostic (nccl on the GPUs, gloo in the CPU tests).
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


def string_range(rank, world, n):
    """CARP string of rank `rank` of `world` (R27): histories [floor(rank n / world), floor((rank + 1) n / world))."""
    if not (0 <= rank < world) or n < world:
        raise ValueError("0 <= rank < world <= n required")
    return (rank * n) // world, ((rank + 1) * n) // world


def carp_distributed(sweep, get_image, set_image, n_iter, world):
    """n_iter CARP iterations with ONE STRING PER RANK (R27-R29).

    sweep()        one DROP sweep of this rank over its own string, from the image it currently holds
    get_image()    -> the rank's image as a tensor (on the device the process group reduces on)
    set_image(t)   makes t the rank's image
    Every rank starts from the same image and ends every iteration with the same one: the arithmetic mean
    of the `world` string solutions, the all-reduce being the method's only exchange."""
    for _ in range(int(n_iter)):
        sweep()
        x = get_image()
        if world > 1:
            dist.all_reduce(x, op=dist.ReduceOp.SUM)
            x /= world
        set_image(x)


class _DeviceArray:
    """A borrowed device array as something torch.as_tensor understands (no copy)."""

    def __init__(self, address, n):
        self.__cuda_array_interface__ = {"shape": (int(n),), "typestr": "<f4", "data": (int(address), False), "version": 3}


def carp_distributed_pct(pct, ctx, n_voxels, lam, block_size, n_iter, world, ctx_stream=None, tvs=False):
    """carp_distributed on a libpct context holding this rank's string (pct = the binding module).

    The average is taken IN PLACE on the library's own image array (pct_image_storage: the storage order is the same
    on every rank of the same grid, and a sum does not care about order): no copy, no host synchronisation.  All of it
    is ordered on the context's stream: ctx_stream is the cudaStream_t handle given to pct_create (None: the context was
    created on torch's current stream), and the collective and the division run under that stream, so the sweep, the
    all-reduce and the next sweep follow one another on the device.

    TVS (pct_set_tvs).  PAPER.md:113: "In CARP, TVS is applied just once to the initial solution at the start of each
    iteration" -- not before every block, which is where pct_iterate puts it (the DROP placement).  With tvs=True the
    rank's sweep is pct_iterate_carp(ctx, ..., n_iter=1, n_strings=1): one TVS step on the common image the iteration
    starts from (the same image, hence the same step, on every rank), then the string's DROP sweep without further
    steps -- the placement of the single-GPU pct_iterate_carp.  With tvs=False (the default) the sweep is pct_iterate
    and the context's TVS must be off; a context with TVS on would take a step before every block of its string."""
    address, n_slots = pct.pct_image_storage(ctx)
    x = torch.as_tensor(_DeviceArray(address, n_slots), device="cuda")
    stream = torch.cuda.current_stream() if ctx_stream is None else torch.cuda.ExternalStream(int(ctx_stream))
    if tvs:
        def sweep():
            pct.pct_iterate_carp(ctx, lam, block_size, 1, 1)
    else:
        def sweep():
            pct.pct_iterate(ctx, lam, block_size, 1)
    with torch.cuda.stream(stream):
        carp_distributed(sweep, lambda: x, lambda t: None, n_iter, world)
