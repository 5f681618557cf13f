"""Host-side logic of the multi-GPU launch (one process per GPU, `torch.distributed`): how the spatial
batch is split and how per-rank timings become one number.  No arithmetic of the method lives here.

dgfs_collide needs no collective: every (spatial point, pair) evaluation is independent
and the paper itself distributes spatial elements linearly over ranks; the tables are replicated.
"""
import torch
import torch.distributed as dist


def shard_range(nx: int, world: int, rank: int):
    """Contiguous block [lo, hi) of `nx` spatial points owned by `rank` (sizes differ by at most one)."""
    if not (0 <= rank < world):
        raise ValueError("rank %d outside world of %d" % (rank, world))
    base, rem = divmod(nx, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def rank_seed(seed: int, rank: int) -> int:
    """Weak scaling: every rank draws its own nx points from its own seed."""
    return seed + 1000 * rank


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of one number (a device-timed duration); identity without a process group."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    if device is None:
        device = torch.device("cuda", torch.cuda.current_device()) if dist.get_backend() == "nccl" else torch.device("cpu")
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank: int, world: int, ms_max: float) -> float:
    """Units all ranks processed per second, with the slowest rank's time."""
    return units_per_rank * world / (ms_max * 1e-3)
