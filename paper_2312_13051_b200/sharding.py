"""Multi-GPU sharding of the path: every Wilson loop is independent, so loops are
partitioned across ranks with no data-path collective; only the (tiny) phase arrays are gathered
at the end.  Host logic only -- shared by bench.py and the world_size-2 gloo test."""
from __future__ import annotations


def shard_range(n_items: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous, balanced [lo, hi) slice of ``n_items`` for ``rank`` (sizes differ by <= 1)."""
    if world < 1 or not (0 <= rank < world) or n_items < 0:
        raise ValueError("bad shard arguments")
    base, rem = divmod(n_items, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def gather_phases(local, n_total: int, rank: int, world: int, group=None):
    """All-gather per-rank phase blocks [n_local][m] into [n_total][m] (torch.distributed)."""
    import torch
    import torch.distributed as dist
    if world == 1:
        return local
    m = local.shape[1]
    sizes = [shard_range(n_total, r, world) for r in range(world)]
    pad = max(hi - lo for lo, hi in sizes)
    buf = torch.zeros((pad, m), dtype=local.dtype, device=local.device)
    buf[: local.shape[0]] = local
    out = [torch.empty_like(buf) for _ in range(world)]
    dist.all_gather(out, buf, group=group)
    return torch.cat([out[r][: sizes[r][1] - sizes[r][0]] for r in range(world)], dim=0)
