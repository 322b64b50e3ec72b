"""Multi-GPU split of the path ("geometry calculations are independent of
each other").  Tracks shard across ranks as contiguous ranges with NO data-path collective; shape constants and
the daughter table are replicated by creating the handles on every rank.  The only communication is the
measurement plumbing below (a barrier and a MAX over ranks of the timed duration)."""
import torch
import torch.distributed as dist


def track_range(n, rank, world):
    """Contiguous range [lo, hi) of rank `rank` out of `world` over n tracks: [n*g/G, n*(g+1)/G)."""
    if not (0 <= rank < world):
        raise ValueError("rank %r outside [0, %r)" % (rank, world))
    return (n * rank) // world, (n * (rank + 1)) // world


def barrier():
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def max_over_ranks(value, device="cpu"):
    """MAX over ranks of a python float (the timed duration); identity without a process group."""
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value, device="cpu"):
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())
