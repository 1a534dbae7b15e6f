"""Host logic of the multi-GPU path: shell quartets are independent units, so ranks take disjoint
contiguous ranges and never exchange integrals.  The only collective is the
MAX reduction of the timed region that bench.py reports."""


def shard_range(n, rank, world):
    """Contiguous, balanced [lo, hi) of n units for `rank` of `world` (sizes differ by at most 1)."""
    if world < 1 or not 0 <= rank < world or n < 0:
        raise ValueError("bad shard arguments")
    base, rem = divmod(n, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def max_over_ranks(value, device="cpu"):
    """MAX of a Python float over the ranks of the default process group (identity without one)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
