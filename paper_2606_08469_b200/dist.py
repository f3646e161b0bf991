"""Multi-GPU plumbing: the path shards trivially — queries are independent, the cache is read-only and
replicated — so there is no data-path collective.  These helpers only split work and reduce timings."""
from __future__ import annotations

import os


def env_rank_world():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def shard_range(n: int, rank: int, world: int):
    """Contiguous slice [lo, hi) of n items for this rank; sizes differ by at most one."""
    base, rem = divmod(n, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def init_process_group(backend: str):
    import torch.distributed as dist
    if not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group(backend=backend)
    return dist


def reduce_max_sum(values_max, values_sum, device):
    """(max over ranks of each entry of values_max, sum over ranks of each entry of values_sum)."""
    import torch
    import torch.distributed as dist
    a = torch.tensor(list(values_max), dtype=torch.float64, device=device)
    b = torch.tensor(list(values_sum), dtype=torch.float64, device=device)
    if dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(a, op=dist.ReduceOp.MAX)
        dist.all_reduce(b, op=dist.ReduceOp.SUM)
    return a.tolist(), b.tolist()
