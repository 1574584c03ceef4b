"""Multi-GPU plumbing: patch groups are independent given padded inputs, so a batch is
sharded by contiguous group ranges (the paper orders patches along a Hilbert curve, L262) with no collective
on the data path; the only exchange is the reduction of one scalar, the time-step (max is order-independent,
so the result stays bitwise reproducible, L178-184)."""
import torch
import torch.distributed as dist


def shard_range(n_groups: int, rank: int, world: int):
    """Contiguous [lo, hi) range of rank `rank`; sizes differ by at most one group."""
    base, rem = divmod(n_groups, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def global_dt(dt: torch.Tensor) -> torch.Tensor:
    """In-place MIN all-reduce of the 1-element dt tensor across ranks (no-op without a process group)."""
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(dt, op=dist.ReduceOp.MIN)
    return dt
