"""Multi-GPU plumbing for the walk: walker-range partition and the one
exchange step, a variable-length all-gather of compacted samples.  Works on any
torch.distributed backend (nccl on GPUs, gloo in the CPU tests); no arithmetic of the method."""
from __future__ import annotations

import torch
import torch.distributed as dist


def walker_range(rank: int, world: int, num_walkers: int) -> tuple[int, int]:
    """Contiguous strong-scaling split of walkers 0..num_walkers-1: (begin, count) of `rank`."""
    base, rem = divmod(num_walkers, world)
    begin = rank * base + min(rank, rem)
    return begin, base + (1 if rank < rem else 0)


def gather_compacted(samples: torch.Tensor, count: int, group=None) -> torch.Tensor:
    """All ranks pass their compacted (count, 12) samples; every rank gets the concatenation in
    rank order (= walker order when ranks hold walker_range()s)."""
    world = dist.get_world_size(group)
    dev = samples.device
    counts = [torch.zeros(1, dtype=torch.int64, device=dev) for _ in range(world)]
    dist.all_gather(counts, torch.tensor([count], dtype=torch.int64, device=dev), group=group)
    counts = [int(c.item()) for c in counts]
    cap = max(max(counts), 1)
    mine = torch.zeros((cap, 12), dtype=torch.float64, device=dev)
    mine[:count] = samples[:count]
    parts = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(parts, mine, group=group)
    return torch.cat([p[:c] for p, c in zip(parts, counts)], dim=0)
