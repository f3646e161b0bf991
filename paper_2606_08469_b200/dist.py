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


def all_gather_rows(local, n_total: int):
    """The one optional collective of the path: every rank computed RGB for its shard_range slice of the
    n_total queries; returns the whole [n_total, C] frame on every rank (NCCL on GPUs: 12 B x N over NVLink; gloo on CPU).
    `local` is this rank's [hi - lo, C] tensor.  With one rank it is returned as is."""
    import torch
    import torch.distributed as dist
    if not dist.is_initialized() or dist.get_world_size() == 1:
        assert local.shape[0] == n_total
        return local
    world, rank = dist.get_world_size(), dist.get_rank()
    lo, hi = shard_range(n_total, rank, world)
    assert local.shape[0] == hi - lo, "local rows %d != this rank's shard %d" % (local.shape[0], hi - lo)
    # shards differ by at most one row: gather equal-sized padded blocks, then drop the padding
    m = -(-n_total // world)
    tail = tuple(local.shape[1:])
    mine = torch.zeros((m,) + tail, dtype=local.dtype, device=local.device)
    mine[: hi - lo] = local
    blocks = torch.empty((world, m) + tail, dtype=local.dtype, device=local.device)
    dist.all_gather([blocks[r] for r in range(world)], mine)      # equal-sized views of one buffer (works on nccl and gloo)
    out = torch.empty((n_total,) + tail, dtype=local.dtype, device=local.device)
    for r in range(world):
        a, b = shard_range(n_total, r, world)
        out[a:b] = blocks[r, : b - a]
    return out
