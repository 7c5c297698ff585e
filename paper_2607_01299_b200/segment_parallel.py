"""Segment parallelism on devices (section 4.4): orchestration only.

One request's cold segments are LPT-sharded over the ranks (Eq. 9, ``sharding.lpt_partition``); every rank encodes its
own segments for all heads with ``hypic_segment_encode`` ("needs no collective communication"), the
tuples ``(T_C, S_{C|0})`` make one all-to-all from the segment-sharded to the head-sharded layout
(``sharding.exchange_tuples``), and every rank folds its heads with ``hypic_compose``.  Finalize-and-ship
(PAPER.md:265-267): a rank's segments are encoded in ``n_groups`` calls, longest first; the exchange of a finished
group runs on a side stream while the next group is encoded.

No arithmetic of the method lives here: the two library calls do all of it.
"""
from __future__ import annotations

import dataclasses
from typing import List, Optional, Sequence

import torch

from . import sharding
from .workloads import EncodeInputs


def take_segments(inp: EncodeInputs, seg_ids: Sequence[int]) -> EncodeInputs:
    """The packed inputs of the given segments only (rows gathered in the order of ``seg_ids``); pure indexing."""
    cu = [0]
    for l in inp.seg_lens:
        cu.append(cu[-1] + int(l))
    if len(seg_ids) == 0:
        idx = torch.empty(0, dtype=torch.long, device=inp.k.device)
    else:
        idx = torch.cat([torch.arange(cu[s], cu[s + 1], device=inp.k.device) for s in seg_ids])
    lens = [int(inp.seg_lens[s]) for s in seg_ids]
    cu_new = torch.zeros(len(lens) + 1, dtype=torch.int32)
    if lens:
        cu_new[1:] = torch.cumsum(torch.tensor(lens, dtype=torch.int64), 0).to(torch.int32)
    return EncodeInputs(k=inp.k[idx].contiguous(), v=inp.v[idx].contiguous(), g=inp.g[idx].contiguous(),
                        beta=inp.beta[idx].contiguous(), cu_seqlens=cu_new.to(inp.k.device), gate=inp.gate, seg_lens=lens)


def split_groups(seg_ids: Sequence[int], seg_lens: Sequence[int], n_groups: int) -> List[List[int]]:
    """A rank's segments in ``n_groups`` batches of similar token count, longest segments first (they finish first and
    ship first); every batch in ascending index order.  Empty batches are allowed (all ranks make ``n_groups`` calls)."""
    order = sorted(seg_ids, key=lambda i: (-int(seg_lens[i]), i))
    groups: List[List[int]] = [[] for _ in range(n_groups)]
    loads = [0] * n_groups
    for i in order:
        g = min(range(n_groups), key=lambda j: (loads[j], j))
        groups[g].append(i)
        loads[g] += int(seg_lens[i])
    return [sorted(g) for g in groups]


@dataclasses.dataclass
class SegmentParallelResult:
    S: torch.Tensor              # [R, Hr, dv, dk]: this rank's heads of the composed state
    head_begin: int
    head_end: int
    exchanged_bytes: int         # bytes this rank sent to OTHER ranks
    E: torch.Tensor              # [n_seg, Hr, dv, dk] pools after the exchange
    T: torch.Tensor


def encode_exchange_compose(hb, my: Sequence[EncodeInputs], groups_all: Sequence[Sequence[Sequence[int]]], n_seg: int,
                            rank: int, world: int, seg_ids: torch.Tensor, cu_segs: torch.Tensor, *,
                            S_in: Optional[torch.Tensor] = None, group=None, via_host: bool = False,
                            comm_stream: Optional[torch.cuda.Stream] = None) -> SegmentParallelResult:
    """``my[g]``: this rank's inputs of group ``g`` (``take_segments``); ``groups_all[g][r]``: the segment ids rank ``r``
    encodes in group ``g`` (every rank derives the same lists).  Encode group g -> ship group g (side stream) while
    group g + 1 encodes -> compose this rank's heads over all ``n_seg`` segments."""
    dev = my[0].k.device
    H, dk, dv = my[0].H, my[0].dk, my[0].dv
    hb_, he_ = sharding.head_range(H, rank, world)
    Hr = he_ - hb_
    E = torch.empty((n_seg, Hr, dv, dk), dtype=torch.float32, device=dev)
    T = torch.empty((n_seg, Hr, dk, dk), dtype=torch.float32, device=dev)
    main = torch.cuda.current_stream(dev)
    comm = comm_stream if comm_stream is not None else torch.cuda.Stream(dev)
    sent = 0
    keep = []
    for g, inp in enumerate(my):
        if inp.n_seg > 0:
            E_loc, T_loc = hb.hypic_segment_encode(inp.k, inp.v, inp.g, inp.beta, inp.cu_seqlens, inp.gate)
        else:
            E_loc = torch.empty((0, H, dv, dk), dtype=torch.float32, device=dev)
            T_loc = torch.empty((0, H, dk, dk), dtype=torch.float32, device=dev)
        done = torch.cuda.Event()
        done.record(main)
        keep.append((E_loc, T_loc))
        E_loc.record_stream(comm)
        T_loc.record_stream(comm)
        with torch.cuda.stream(comm):
            comm.wait_event(done)  # the group is final: ship it while the next one is encoded on the main stream
            sharding.exchange_tuples(E_loc, T_loc, groups_all[g], rank, world, group=group, out=(E, T), n_seg=n_seg,
                                     via_host=via_host)
        sent += inp.n_seg * (H - Hr) * (dv * dk + dk * dk) * 4
    main.wait_stream(comm)
    S = hb.hypic_compose(None if S_in is None else S_in[:, hb_:he_].contiguous(), E, T, seg_ids, cu_segs)
    return SegmentParallelResult(S=S, head_begin=hb_, head_end=he_, exchanged_bytes=sent, E=E, T=T)


def plan(seg_lens: Sequence[int], world: int, n_groups: int):
    """(parts, groups_all): LPT partition of the segments over the ranks, and each rank's share cut into groups."""
    parts = sharding.lpt_partition(seg_lens, world)
    per_rank = [split_groups(parts[r], seg_lens, n_groups) for r in range(world)]
    groups_all = [[per_rank[r][g] for r in range(world)] for g in range(n_groups)]
    return parts, groups_all
