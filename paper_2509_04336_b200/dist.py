"""Multi-GPU plumbing: one process per GPU, rows / walker slots sharded, no data-path collective.

torch.distributed is used for the timing barrier and the max-over-ranks reduction only.  The Philox streams are keyed by the
global row / walker slot, so a sharded run computes exactly the rows a single-GPU run would (any partition, same results)."""
import os

import torch
import torch.distributed as dist


def env():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0"))


def init(backend=None, device=None):
    rank, world, local = env()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        if backend is None:
            backend = "nccl" if torch.cuda.is_available() else "gloo"
        kw = {"device_id": device} if (backend == "nccl" and device is not None) else {}
        dist.init_process_group(backend, **kw)
    return rank, world, local


def shard_range(n, rank, world):
    """Contiguous slot range [lo, hi) of rank `rank` when n walker slots / rows are split over `world` ranks
    (slot j goes to rank floor(j * world / n)'s inverse: lo = ceil(rank n / world))."""
    lo = (rank * n + world - 1) // world
    hi = ((rank + 1) * n + world - 1) // world
    return lo, hi


def barrier(device=None):
    if dist.is_initialized():
        dist.barrier()
    if device is not None and torch.cuda.is_available():
        torch.cuda.synchronize()


def max_over_ranks(x, device="cpu"):
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    if dist.is_initialized():
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x, device="cpu"):
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    if dist.is_initialized():
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def finalize():
    if dist.is_initialized():
        dist.destroy_process_group()
