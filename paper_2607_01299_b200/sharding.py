"""Host-side sharding of the hot path across GPUs (one process per GPU): no arithmetic of the method lives here.

The path shards by independent units: segments for encode ("needs no collective
communication"), (request, head) chains for compose.  There is no data-path collective; the only
communication is the timing reduction (max over ranks) that bench.py reports.

* ``lpt_partition`` -- the paper's longest-processing-time assignment of cold segments to workers
  (Eq. 9: min over assignments of the max per-worker token count).
* ``head_range`` -- contiguous split of the head axis for compose-only workloads.
* ``max_over_ranks`` -- device- or host-side MAX all-reduce of a timing, on whatever backend the group uses.
"""
from __future__ import annotations

import heapq
from typing import List, Optional, Sequence, Tuple

import torch


def lpt_partition(seg_lens: Sequence[int], world_size: int) -> List[List[int]]:
    """Segments sorted by length (descending, ties by index) are given one by one to the least-loaded worker.
    Returns, per worker, the segment indices it owns (in ascending index order).  Deterministic, so every rank
    computes the same partition without talking to the others."""
    if world_size <= 0:
        raise ValueError("world_size must be positive")
    order = sorted(range(len(seg_lens)), key=lambda i: (-int(seg_lens[i]), i))
    heap: List[Tuple[int, int]] = [(0, w) for w in range(world_size)]
    heapq.heapify(heap)
    owned: List[List[int]] = [[] for _ in range(world_size)]
    for i in order:
        load, w = heapq.heappop(heap)
        owned[w].append(i)
        heapq.heappush(heap, (load + int(seg_lens[i]), w))
    return [sorted(o) for o in owned]


def shard_loads(seg_lens: Sequence[int], parts: Sequence[Sequence[int]]) -> List[int]:
    return [sum(int(seg_lens[i]) for i in p) for p in parts]


def head_range(n_heads: int, rank: int, world_size: int) -> Tuple[int, int]:
    """[begin, end) of the heads rank owns when the head axis is split as evenly as possible."""
    base, rem = divmod(n_heads, world_size)
    begin = rank * base + min(rank, rem)
    return begin, begin + base + (1 if rank < rem else 0)


def max_over_ranks(value: float, device: Optional[torch.device] = None, group=None) -> float:
    """MAX all-reduce of one number (multi-GPU timings are the max over ranks, never a wall clock)."""
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())
