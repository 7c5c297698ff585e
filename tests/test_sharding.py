"""N > 1 host logic on CPU: LPT segment partition (Eq. 9), head split, and the max-over-ranks
timing reduction over a world_size-2 gloo group.  Also: encoding a shard of the segments and composing per head
with the oracle gives the same state as the unsharded run (the path shards with no data-path collective)."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
from paper_2607_01299_b200 import segment_parallel as sp
from paper_2607_01299_b200 import sharding
from paper_2607_01299_b200 import workloads as wl


def test_lpt_partition_covers_and_balances():
    lens = wl.cfg3_seg_lens()
    for world in (1, 2, 3, 8):
        parts = sharding.lpt_partition(lens, world)
        assert sorted(i for p in parts for i in p) == list(range(len(lens)))
        loads = sharding.shard_loads(lens, parts)
        # greedy list scheduling: the fullest worker, minus the last segment it was given, is no fuller than the mean
        assert max(loads) <= sum(lens) / world + max(lens)
        if world == 1:
            assert loads == [sum(lens)]
    assert sharding.lpt_partition([], 4) == [[], [], [], []]
    assert sharding.lpt_partition([5, 5, 5], 2) == [[0, 2], [1]]


def test_head_range_is_a_partition():
    for H in (1, 16, 32, 33):
        for world in (1, 2, 3, 8):
            spans = [sharding.head_range(H, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == H
            assert all(spans[i][1] == spans[i + 1][0] for i in range(world - 1))
            sizes = [e - b for b, e in spans]
            assert max(sizes) - min(sizes) <= 1


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir, H=2):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        inp = wl.make_encode_inputs([70, 33, 129, 64, 5], H, 16, 16, kv_dtype=torch.float32, seed=wl.seed_for(0, 9))
        parts = sharding.lpt_partition(inp.seg_lens, world)
        mine = parts[rank]
        # every rank derives the same partition on its own
        gathered = [None] * world
        dist.all_gather_object(gathered, parts)
        assert all(g == parts for g in gathered)
        # encode my segments only (oracle stands in for the device on the CPU box); no collective on the data path
        E_all, T_all = oracle.segment_encode(inp.k, inp.v, inp.g, inp.beta, inp.cu_seqlens, gate=inp.gate)
        cu = inp.cu_seqlens.numpy()
        for s in mine:
            sl = slice(int(cu[s]), int(cu[s + 1]))
            E, T = oracle.segment_encode(inp.k[sl], inp.v[sl], inp.g[sl], inp.beta[sl],
                                         np.array([0, sl.stop - sl.start], dtype=np.int32), gate=inp.gate)
            assert np.array_equal(E[0], E_all[s]) and np.array_equal(T[0], T_all[s])
        # compose is sharded by heads: my heads of the composed state equal the same heads of the full run
        b, e = sharding.head_range(H, rank, world)
        ids = np.arange(5, dtype=np.int32)
        cu_r = np.array([0, 5], dtype=np.int32)
        S_full = oracle.compose(None, E_all, T_all, ids, cu_r)
        S_mine = oracle.compose(None, E_all[:, b:e], T_all[:, b:e], ids, cu_r)
        assert np.array_equal(S_mine, S_full[:, b:e])
        # the exchange step of segment parallelism: my segments x all heads -> all segments x my heads, one all-to-all
        E_loc = torch.from_numpy(np.ascontiguousarray(E_all[mine]))
        T_loc = torch.from_numpy(np.ascontiguousarray(T_all[mine]))
        E_x, T_x = sharding.exchange_tuples(E_loc, T_loc, parts, rank, world)
        assert torch.equal(E_x, torch.from_numpy(np.ascontiguousarray(E_all[:, b:e])))
        assert torch.equal(T_x, torch.from_numpy(np.ascontiguousarray(T_all[:, b:e])))
        S_x = oracle.compose(None, E_x.numpy(), T_x.numpy(), ids, cu_r)
        assert np.array_equal(S_x, S_full[:, b:e])
        # timing reduction: max over ranks
        t = sharding.max_over_ranks(10.0 + rank)
        assert t == 10.0 + world - 1
        with open(os.path.join(out_dir, f"ok{rank}"), "w") as f:
            f.write("ok")
    finally:
        dist.destroy_process_group()


def test_exchange_tuples_single_rank_is_a_reorder():
    E = torch.arange(3 * 2 * 4 * 4, dtype=torch.float32).reshape(3, 2, 4, 4)
    T = -E.clone()
    parts = [[0, 1, 2]]
    E_x, T_x = sharding.exchange_tuples(E, T, parts, 0, 1)
    assert torch.equal(E_x, E) and torch.equal(T_x, T)


def test_two_rank_gloo_sharding(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    assert all((tmp_path / f"ok{r}").exists() for r in range(world))


def test_three_rank_gloo_uneven_heads(tmp_path):
    """3 ranks, 4 heads (2 + 1 + 1) and 5 segments (LPT gives 2 + 2 + 1): uneven on both axes of the all-to-all."""
    world = 3
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path), 4), nprocs=world, join=True)
    assert all((tmp_path / f"ok{r}").exists() for r in range(world))


def test_fold_layers_is_a_pure_relayout():
    """fold_layers: head l*H + h of the folded inputs is head h of layer l, bit for bit; the oracle on a folded unit
    equals the oracle on the layer's own unit (layers stay independent)."""
    layers = [wl.make_encode_inputs([70, 33], 2, 16, 16, kv_dtype=torch.float32, seed=wl.seed_for(0, 40 + l))
              for l in range(3)]
    f = wl.fold_layers(layers)
    assert f.H == 6 and f.seg_lens == [70, 33] and f.k.is_contiguous()
    for l, x in enumerate(layers):
        for name in ("k", "v", "g", "beta"):
            assert torch.equal(getattr(f, name)[:, 2 * l:2 * l + 2], getattr(x, name))
    Ef, Tf = oracle.segment_encode(f.k.numpy(), f.v.numpy(), f.g.numpy(), f.beta.numpy(), f.cu_seqlens.numpy())
    E1, T1 = oracle.segment_encode(layers[1].k.numpy(), layers[1].v.numpy(), layers[1].g.numpy(), layers[1].beta.numpy(),
                           layers[1].cu_seqlens.numpy())
    assert np.array_equal(Ef[:, 2:4], E1) and np.array_equal(Tf[:, 2:4], T1)



# ------------------------------------------------------------------ segment parallelism: plan, groups, grouped exchange
def test_plan_groups_cover_every_segment_once():
    lens = wl.cfg3_seg_lens()
    for world in (1, 2, 3):
        for n_groups in (1, 2, 4):
            parts, groups_all = sp.plan(lens, world, n_groups)
            assert len(groups_all) == n_groups and all(len(g) == world for g in groups_all)
            for r in range(world):
                mine = sorted(i for g in groups_all for i in g[r])
                assert mine == parts[r]
            # longest first: the first group of a rank holds its longest segment
            for r in range(world):
                if parts[r]:
                    longest = max(parts[r], key=lambda i: (lens[i], -i))
                    assert longest in groups_all[0][r]


def test_take_segments_is_pure_indexing():
    inp = wl.make_encode_inputs([7, 0, 5, 9], 2, 8, 8, kv_dtype=torch.float32, seed=3)
    sub = sp.take_segments(inp, [3, 0])
    assert sub.seg_lens == [9, 7] and sub.cu_seqlens.tolist() == [0, 9, 16]
    assert torch.equal(sub.k[:9], inp.k[12:21]) and torch.equal(sub.k[9:], inp.k[:7])
    assert torch.equal(sub.g[:9], inp.g[12:21]) and torch.equal(sub.beta[9:], inp.beta[:7])
    empty = sp.take_segments(inp, [])
    assert empty.n_seg == 0 and empty.t_total == 0


def _worker_groups(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        H = 3
        inp = wl.make_encode_inputs([70, 33, 129, 64, 5, 90], H, 16, 16, kv_dtype=torch.float32, seed=wl.seed_for(0, 11))
        E_all, T_all = oracle.segment_encode(inp.k, inp.v, inp.g, inp.beta, inp.cu_seqlens, gate=inp.gate)
        parts, groups_all = sp.plan(inp.seg_lens, world, 3)
        b, e = sharding.head_range(H, rank, world)
        E = torch.full((6, e - b, 16, 16), float("nan"))
        T = torch.full((6, e - b, 16, 16), float("nan"))
        for g in range(3):  # one exchange per finished group, all filling the same pools
            mine = groups_all[g][rank]
            E_loc = torch.from_numpy(np.ascontiguousarray(E_all[mine])).float().reshape(len(mine), H, 16, 16)
            T_loc = torch.from_numpy(np.ascontiguousarray(T_all[mine])).float().reshape(len(mine), H, 16, 16)
            sharding.exchange_tuples(E_loc, T_loc, groups_all[g], rank, world, out=(E, T), n_seg=6)
        assert torch.equal(E, torch.from_numpy(np.ascontiguousarray(E_all[:, b:e])).float())
        assert torch.equal(T, torch.from_numpy(np.ascontiguousarray(T_all[:, b:e])).float())
        with open(os.path.join(out_dir, f"ok{rank}"), "w") as f:
            f.write("ok")
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_grouped_exchange(tmp_path):
    """Finalize-and-ship: three exchanges, one per finished group (one of them empty on a rank), assemble
    the same head-sharded pools as the single all-to-all."""
    world = 2
    mp.spawn(_worker_groups, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    assert all((tmp_path / f"ok{r}").exists() for r in range(world))
