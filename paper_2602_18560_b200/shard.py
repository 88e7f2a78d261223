"""Host-side sharding of independent catalogs over ranks.

The path shards by independent problems only: every catalog of a batch (config 4: 64 of them) runs to its
own convergence, so catalogs are dealt to ranks and no collective touches the data path.  What is
exchanged is bookkeeping: the per-catalog outcomes gathered on rank 0 and the max-over-ranks step time.
One process per GPU; `torch.distributed` (NCCL on GPUs, gloo in the CPU tests) is the plumbing.
"""
from __future__ import annotations

from typing import Dict, List, Sequence


def partition_catalogs(n_src: Sequence[int], world_size: int) -> List[List[int]]:
    """Deals catalog ids to ranks, balancing the number of sources (longest processing time first:
    cost of a catalog ~ its source count).  Deterministic: ties go to the lower rank, ids of a rank are
    returned in increasing order.  Every id appears exactly once."""
    if world_size < 1:
        raise ValueError("world_size must be >= 1")
    order = sorted(range(len(n_src)), key=lambda c: (-int(n_src[c]), c))
    load = [0] * world_size
    parts: List[List[int]] = [[] for _ in range(world_size)]
    for c in order:
        r = min(range(world_size), key=lambda k: (load[k], k))
        parts[r].append(c)
        load[r] += int(n_src[c])
    return [sorted(p) for p in parts]


def local_offsets(n_src: Sequence[int], cat_ids: Sequence[int]) -> List[int]:
    """`offsets` ([len+1], offsets[0] = 0) of the concatenation of the given catalogs (include/gbfg.h)."""
    off = [0]
    for c in cat_ids:
        off.append(off[-1] + int(n_src[c]))
    return off


def max_over_ranks(value: float, device=None, group=None) -> float:
    """Step time of the job = the slowest rank's."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())


def gather_outcomes(local: Dict[int, dict], group=None) -> Dict[int, dict]:
    """Per-catalog outcomes {catalog id: {...}} of every rank, merged (on every rank).  A catalog reported by
    two ranks is a partition bug and raises."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return dict(local)
    parts = [None] * dist.get_world_size(group)
    dist.all_gather_object(parts, dict(local), group=group)
    merged: Dict[int, dict] = {}
    for p in parts:
        for c, v in p.items():
            if c in merged:
                raise RuntimeError(f"catalog {c} was processed by two ranks")
            merged[c] = v
    return merged
