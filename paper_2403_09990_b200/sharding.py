"""Multi-GPU plumbing for the walk: walker-range partition and the one
exchange step of a sharded instance, a variable-length gather of compacted samples on the rank
that runs the miniball.  Works on any torch.distributed backend (nccl on GPUs, gloo in the CPU
tests); no arithmetic of the method."""
from __future__ import annotations

import torch
import torch.distributed as dist


def walker_range(rank: int, world: int, num_walkers: int) -> tuple[int, int]:
    """Contiguous strong-scaling split of walkers 0..num_walkers-1: (begin, count) of `rank`."""
    base, rem = divmod(num_walkers, world)
    begin = rank * base + min(rank, rem)
    return begin, base + (1 if rank < rem else 0)


def gather_counts(count: int, device, group=None) -> list[int]:
    """Every rank's number of compacted samples, on every rank (one 8-byte all-gather)."""
    world = dist.get_world_size(group)
    mine = torch.tensor([count], dtype=torch.int64, device=device)
    out = torch.empty((world,), dtype=torch.int64, device=device)
    dist.all_gather_into_tensor(out, mine, group=group)
    return [int(c) for c in out.tolist()]


def gather_to_root(samples: torch.Tensor, count: int, root: int = 0, group=None):
    """The exchange step: rank r passes its compacted (count, 12) samples; `root` gets the
    concatenation in rank order (= walker order when ranks hold walker_range()s), the others get None.
    Nothing is padded: the counts are gathered first, the root sizes one buffer from them and every other
    rank sends exactly its count x 96 bytes point to point into the root's slice."""
    rank = dist.get_rank(group)
    counts = gather_counts(count, samples.device, group)
    total = sum(counts)
    if rank == root:
        merged = torch.empty((total, 12), dtype=samples.dtype, device=samples.device)
        offs, ops = 0, []
        for r, c in enumerate(counts):
            if r == root:
                merged[offs:offs + c] = samples[:c]
            elif c > 0:
                ops.append(dist.P2POp(dist.irecv, merged[offs:offs + c], r, group=group))
            offs += c
        if ops:
            for req in dist.batch_isend_irecv(ops):
                req.wait()
        return merged, counts
    if count > 0:
        for req in dist.batch_isend_irecv([dist.P2POp(dist.isend, samples[:count].contiguous(), root, group=group)]):
            req.wait()
    return None, counts


def gather_compacted(samples: torch.Tensor, count: int, group=None) -> torch.Tensor:
    """All ranks get the concatenation (rank order) of every rank's compacted samples: gather on rank 0, then one
    broadcast of the merged cloud -- for callers that want the cloud everywhere; the walk itself only needs
    gather_to_root."""
    merged, counts = gather_to_root(samples, count, 0, group)
    if dist.get_rank(group) != 0:
        merged = torch.empty((sum(counts), 12), dtype=samples.dtype, device=samples.device)
    if merged.shape[0] > 0:
        dist.broadcast(merged, 0, group=group)
    return merged


def strong_step(sample, compact, megb, num_walkers: int, rank: int, world: int, root: int = 0, group=None,
                device=None):
    """One strong-scaling step of ONE instance over `world` ranks (bench.py --scaling strong; the gloo test drives
    the same function with the oracle standing in for the device calls):
        sample(begin, n)        -> (samples (n,12), flags (n,))  walkers begin .. begin+n-1 of the instance
        compact(samples, flags) -> (compacted (>=count,12), count tensor)
        megb(cloud, count)      -> result dict, called on `root` only
    Returns megb's result (plus "count", "counts") on the root, None elsewhere."""
    begin, n = walker_range(rank, world, num_walkers)
    if n > 0:
        smp, flg = sample(begin, n)[:2]
        comp, cnt = compact(smp, flg)
        count = int(cnt.item())
    else:
        comp = torch.empty((0, 12), dtype=torch.float64, device=device)    # more ranks than walkers
        count = 0
    merged, counts = gather_to_root(comp, count, root, group)
    if rank != root:
        return None
    total = sum(counts)
    if total == 0:
        return {"count": 0, "counts": counts}
    res = dict(megb(merged, total))
    res["count"] = total
    res["counts"] = counts
    return res
