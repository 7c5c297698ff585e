"""Host-side sharding of the hot path across GPUs (one process per GPU): no arithmetic of the method lives here.

The path shards by independent units: segments for encode ("needs no collective
communication"), (request, head) chains for compose.  There is no data-path collective; the only
communication is the timing reduction (max over ranks) that bench.py reports.

* ``lpt_partition`` -- the paper's longest-processing-time assignment of cold segments to workers
  (Eq. 9: min over assignments of the max per-worker token count).
* ``head_range`` -- contiguous split of the head axis for compose-only workloads.
* ``max_over_ranks`` -- device- or host-side MAX all-reduce of a timing, on whatever backend the group uses.
* ``exchange_tuples`` -- the one real exchange step of segment parallelism (scatter workers
  ship their segments' ``(T_C, S_{C|0})`` to where the state is assembled), in its data-parallel form: encode is sharded
  by segments (LPT), compose by heads, so the tuples make one all-to-all between the two layouts.  Pure data movement
  (``torch.distributed.all_to_all_single`` over NCCL on GPUs, gloo in the CPU tests); no arithmetic.
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


def exchange_tuples(E_loc: torch.Tensor, T_loc: torch.Tensor, parts: Sequence[Sequence[int]], rank: int,
                    world_size: int, group=None, out: Optional[Tuple[torch.Tensor, torch.Tensor]] = None,
                    n_seg: Optional[int] = None, via_host: bool = False) -> Tuple[torch.Tensor, torch.Tensor]:
    """From the segment-sharded layout of encode to the head-sharded layout of compose.

    ``E_loc:[len(parts[rank]), H, dv, dk]`` and ``T_loc:[len(parts[rank]), H, dk, dk]`` are this rank's tuples, rows in
    the order of ``parts[rank]`` (``lpt_partition``'s ascending segment indices).  Returns
    ``(E:[n_seg, Hr, dv, dk], T:[n_seg, Hr, dk, dk])`` for ALL segments in global index order and this rank's heads
    ``head_range(H, rank, world_size)``: exactly the pools ``hypic_compose`` takes with ``H = Hr``.
    One all-to-all; rank ``s`` sends rank ``d`` the block ``[parts[s], heads of d]`` of both tensors.

    ``out = (E, T)`` with ``n_seg`` rows: fill these buffers instead of new ones, so that several calls -- one per
    finished group of segments, ``parts`` then being the group's share of every rank (finalize-and-ship,
    PAPER.md:265-267) -- assemble one pool.  ``via_host``: stage the blocks through host memory (a ``gloo`` group with
    device tensors: ranks that share one GPU in a test cannot form an NCCL communicator)."""
    import torch.distributed as dist

    n_loc, H, dv, dk = (int(x) for x in E_loc.shape)
    if tuple(T_loc.shape) != (n_loc, H, dk, dk) or n_loc != len(parts[rank]):
        raise ValueError("E_loc / T_loc do not match parts[rank]")
    if n_seg is None:
        n_seg = sum(len(p) for p in parts)
    hb, he = head_range(H, rank, world_size)
    Hr = he - hb
    per_head = dv * dk + dk * dk
    if out is not None:
        E, T = out
        if tuple(E.shape) != (n_seg, Hr, dv, dk) or tuple(T.shape) != (n_seg, Hr, dk, dk):
            raise ValueError("out buffers must be [n_seg, Hr, dv, dk] and [n_seg, Hr, dk, dk]")
    else:
        E = torch.empty((n_seg, Hr, dv, dk), dtype=E_loc.dtype, device=E_loc.device)
        T = torch.empty((n_seg, Hr, dk, dk), dtype=E_loc.dtype, device=E_loc.device)
    if world_size == 1:
        order = torch.as_tensor(list(parts[0]), dtype=torch.long, device=E_loc.device)
        E[order], T[order] = E_loc, T_loc
        return E, T
    send_chunks, send_sizes = [], []
    for d in range(world_size):
        b, e = head_range(H, d, world_size)
        blk = torch.cat([E_loc[:, b:e].reshape(n_loc, e - b, dv * dk), T_loc[:, b:e].reshape(n_loc, e - b, dk * dk)],
                        dim=2)  # [n_loc, heads of d, per_head]
        send_chunks.append(blk.reshape(-1))
        send_sizes.append(n_loc * (e - b) * per_head)
    recv_sizes = [len(parts[s]) * Hr * per_head for s in range(world_size)]
    send = torch.cat(send_chunks)
    if via_host:
        send_h = send.cpu()
        recv_h = torch.empty(sum(recv_sizes), dtype=E_loc.dtype)
        dist.all_to_all_single(recv_h, send_h, output_split_sizes=recv_sizes, input_split_sizes=send_sizes, group=group)
        recv = recv_h.to(E_loc.device)
    else:
        recv = torch.empty(sum(recv_sizes), dtype=E_loc.dtype, device=E_loc.device)
        dist.all_to_all_single(recv, send, output_split_sizes=recv_sizes, input_split_sizes=send_sizes, group=group)
    off = 0
    for s in range(world_size):
        n_s = len(parts[s])
        if n_s == 0:
            continue
        blk = recv[off:off + recv_sizes[s]].reshape(n_s, Hr, per_head)
        off += recv_sizes[s]
        idx = torch.as_tensor(list(parts[s]), dtype=torch.long, device=E_loc.device)
        E[idx] = blk[:, :, :dv * dk].reshape(n_s, Hr, dv, dk)
        T[idx] = blk[:, :, dv * dk:].reshape(n_s, Hr, dk, dk)
    return E, T
