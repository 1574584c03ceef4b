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


def _reduce_device() -> torch.device:
    """Where a tensor must live to be all-reduced by the current process group: NCCL reduces device tensors only."""
    if dist.get_backend() == "nccl":
        return torch.device("cuda", torch.cuda.current_device())
    return torch.device("cpu")


def global_count(n) -> int:
    """SUM all-reduce of one integer (e.g. the unphysical-cell count of a rank's shard).  `n` is an int or a 1-element
    integer tensor (the device counter that gamer_fluid_advance_ex filled); the reduction runs on the device the
    backend needs (NCCL: the current CUDA device, gloo: the host)."""
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dev = _reduce_device()
        if torch.is_tensor(n):
            t = n.detach().reshape(1).to(device=dev, dtype=torch.int64)
        else:
            t = torch.tensor([int(n)], dtype=torch.int64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        return int(t.item())
    return int(n.item()) if torch.is_tensor(n) else int(n)


def retry_level(step_fn, dt: float, dt_ratio: float = 0.8, dt_min: float = 0.0, max_retries: int = 200):
    """The DISTRIBUTED form of gamer_fluid_advance_retry (csrc/api.cu), which is its single-process form: the same policy
    (dt multiplied by dt_ratio per retry, threshold test before the attempt, at most 200 reductions; R23) with the
    one thing a single process cannot do, the reduction of the count over ranks between attempts.  tests/test_multirank_cpu.py
    holds the two to the same (dt_used, n_retries) through the oracle's loop.
    Remedies (iv), (v) of PAPER.md L107-108 for a level sharded over ranks: "recalculate ALL patches on the currently
    targeted level with this reduced time-step" -- a rank whose own shard came out physical must redo it too, so the
    decision is taken on the SUM of the ranks' counts.  step_fn(dt) advances this rank's shard from its unchanged input
    (e.g. binding.gamer_fluid_advance_ex with n_unphysical_out) and returns its count of unphysical cells.
    Returns (dt_used, n_retries), identical on every rank and to gamer_fluid_advance_retry on the unsharded batch;
    raises ArithmeticError on every rank when the reduced step falls below dt_min (the paper's abort)."""
    if not (0.0 < dt_ratio < 1.0) or not dt > 0.0 or dt_min < 0.0:
        raise ValueError("need dt > 0, 0 < dt_ratio < 1, dt_min >= 0")
    n = 0
    while True:
        if global_count(step_fn(dt)) == 0:
            return dt, n
        dt = dt * dt_ratio
        n += 1
        if dt < dt_min or n > max_retries:
            raise ArithmeticError(f"unphysical cells remain and the reduced time-step {dt} is below dt_min {dt_min}")
