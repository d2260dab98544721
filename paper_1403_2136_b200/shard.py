"""Multi-GPU host logic: reads are independent units, so they are sharded over ranks with the genome replicated and no
data-path collective ("spreading reads across multiple GPUs").  The only exchanges are
control-plane: the max-over-ranks of the timed region and, when a caller wants the whole result in one place, a gather of the
32-byte records.  Works with any torch.distributed backend (nccl on GPUs, gloo in the CPU tests)."""
from __future__ import annotations


def shard_bounds(n_reads: int, world: int) -> list[int]:
    """world+1 cut points: rank r owns reads [b[r], b[r+1]); sizes differ by at most one, lower ranks take the extra."""
    if n_reads < 0 or world < 1:
        raise ValueError("n_reads >= 0 and world >= 1 required")
    q, rem = divmod(n_reads, world)
    b = [0]
    for r in range(world):
        b.append(b[-1] + q + (1 if r < rem else 0))
    return b


def shard_range(n_reads: int, rank: int, world: int) -> tuple[int, int]:
    b = shard_bounds(n_reads, world)
    return b[rank], b[rank + 1]


def max_over_ranks(value: float, device=None) -> float:
    """Max of a per-rank scalar (the timed region's device milliseconds) over all ranks; identity when not distributed."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def gather_records(local, n_reads: int):
    """All ranks' record tensors (first dim = this rank's reads, in shard order) -> the full (n_reads, ...) tensor on
    every rank.  Shards may differ in size by one, so they are padded to the largest before the all_gather."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return local
    world = dist.get_world_size()
    b = shard_bounds(n_reads, world)
    biggest = max(b[r + 1] - b[r] for r in range(world))
    pad = torch.zeros((biggest,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    pad[: local.shape[0]] = local
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad)
    return torch.cat([parts[r][: b[r + 1] - b[r]] for r in range(world)], dim=0)
