"""Member sharding across GPUs: ensemble members are independent, so E is cut into
contiguous ranges, one per rank; the plan matrices are replicated; dns_step needs NO collective.  Only the
6 E diagnostics doubles (and timings) are gathered.  Host logic only -- works on gloo (CPU) and nccl."""
from __future__ import annotations

import numpy as np


def member_range(E: int, rank: int, world: int) -> range:
    """Contiguous, balanced partition: the first E % world ranks get one extra member."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("bad rank/world")
    q, r = divmod(int(E), world)
    lo = rank * q + min(rank, r)
    return range(lo, lo + q + (1 if rank < r else 0))


def gather_rows(local_rows: np.ndarray, E: int, ncols: int):
    """All ranks receive the [E][ncols] array assembled from every rank's rows (torch.distributed)."""
    import torch
    import torch.distributed as dist

    world, rank = dist.get_world_size(), dist.get_rank()
    counts = [len(member_range(E, r, world)) for r in range(world)]
    mx = max(counts)
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    buf = torch.zeros((mx, ncols), dtype=torch.float64, device=dev)
    buf[: counts[rank]] = torch.as_tensor(np.asarray(local_rows, dtype=np.float64).reshape(counts[rank], ncols))
    out = [torch.zeros_like(buf) for _ in range(world)]
    dist.all_gather(out, buf)
    return np.concatenate([o[:c].cpu().numpy() for o, c in zip(out, counts)], axis=0)


def allreduce_sum_(t) -> None:
    """In-place sum over all ranks of a torch tensor (the exchange step of a coupled ensemble sharded over GPUs,
    SURVEY.md 8(f) row f2): NCCL on the tensor's CUDA stream order, gloo for CPU tensors."""
    import torch.distributed as dist

    dist.all_reduce(t, op=dist.ReduceOp.SUM)


def max_over_ranks(x: float) -> float:
    import torch
    import torch.distributed as dist

    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(x)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
