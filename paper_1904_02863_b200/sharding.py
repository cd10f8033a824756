"""Multi-GPU layout of the hot path: proposals are independent units, so a batch is cut
into contiguous per-rank ranges and every rank evaluates its range against its own replica of the context
tables.  There is no data-path collective; a gather of the per-rank lnL slices is only needed when one rank
wants them all.  Host logic only (used by bench.py and by the world_size-2 gloo test)."""
from __future__ import annotations

from typing import List, Tuple


def shard_range(n_items: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous [lo, hi) of rank's share; sizes differ by at most one, earlier ranks get the extra item."""
    if world < 1 or not (0 <= rank < world) or n_items < 0:
        raise ValueError("bad shard request")
    base, extra = divmod(n_items, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def shard_sizes(n_items: int, world: int) -> List[int]:
    return [shard_range(n_items, r, world)[1] - shard_range(n_items, r, world)[0] for r in range(world)]


def gather_lnl(local_lnl, n_items: int, group=None):
    """all_gather the per-rank lnL slices (torch tensors, any backend) into one [n_items] tensor, in rank order."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)
    sizes = shard_sizes(n_items, world)
    width = max(sizes) if sizes else 0
    pad = torch.zeros(width, dtype=local_lnl.dtype, device=local_lnl.device)
    pad[: local_lnl.numel()] = local_lnl
    bufs = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(bufs, pad, group=group)
    return torch.cat([b[:s] for b, s in zip(bufs, sizes)])


# ---- bin sharding (SURVEY.md 8(e) alternative, NEXT-4): few proposals, long signals ------------------------------
# Every inner product is a sum over bins, so ranks may own contiguous frequency sub-bands instead: each rank builds a
# context on freqs[lo:hi] (still a uniform grid), evaluates parts[B][n_det][3] = (Re<d|h>, Im<d|h>, <h|h>) for ALL
# proposals on its sub-band, and one exchange step sums the parts.  To stay run-to-run deterministic the sum is an
# all_gather followed by additions in rank order on every rank (payload B * n_det * 3 doubles per rank), not a
# tree all-reduce whose order the backend may choose.

def bin_shard_edges(n_bins: int, world: int) -> List[Tuple[int, int]]:
    """Contiguous [lo, hi) bin ranges, one per rank (sizes differ by at most one)."""
    return [shard_range(n_bins, r, world) for r in range(world)]


def reduce_parts_rank_ordered(local_parts, group=None):
    """Sum parts over ranks in rank order (identical bits on every rank).  torch tensors, any backend."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)
    bufs = [torch.empty_like(local_parts) for _ in range(world)]
    dist.all_gather(bufs, local_parts.contiguous(), group=group)
    total = bufs[0].clone()
    for b in bufs[1:]:
        total += b
    return total


def lnl_from_parts(parts):
    """lnL[b] = sum_I (Re<d|h>_I - 1/2 <h|h>_I) from summed parts[B][n_det][3] (torch or numpy)."""
    return (parts[..., 0] - 0.5 * parts[..., 2]).sum(-1)
