"""Segment parallelism on devices: shard -> encode -> exchange -> compose on
the GPU equals the unsharded GPU result bit for bit.  Two processes share the one GPU of the box; the exchange goes
through a gloo group with host staging (two ranks on one device cannot form an NCCL communicator; on a multi-GPU node
the same call runs over NCCL).  The kernels of the two processes never wait on one another."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

pytestmark = pytest.mark.gpu


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from paper_2607_01299_b200 import binding as hb
        from paper_2607_01299_b200 import segment_parallel as sp
        from paper_2607_01299_b200 import workloads as wl
        torch.cuda.set_device(0)
        hb.load_library()
        H = 6
        lens = [700, 64, 1300, 129, 2048, 333, 0, 900]
        inp = wl.make_encode_inputs(lens, H, 128, 128, kv_dtype=torch.bfloat16, seed=wl.seed_for(2, 77), device="cuda")
        n_seg = len(lens)
        ids = torch.arange(n_seg, dtype=torch.int32, device="cuda")
        cu = torch.tensor([0, n_seg], dtype=torch.int32, device="cuda")
        gen = torch.Generator(device="cuda")
        gen.manual_seed(5)
        S_in = torch.randn((1, H, 128, 128), generator=gen, device="cuda", dtype=torch.float32)
        # unsharded reference on this GPU
        E0, T0 = hb.hypic_segment_encode(inp.k, inp.v, inp.g, inp.beta, inp.cu_seqlens, inp.gate)
        S0 = hb.hypic_compose(S_in, E0, T0, ids, cu)
        torch.cuda.synchronize()
        # sharded: LPT over ranks, two groups per rank (finalize-and-ship), all-to-all, head-sharded compose
        parts, groups_all = sp.plan(lens, world, 2)
        my = [sp.take_segments(inp, groups_all[g][rank]) for g in range(2)]
        res = sp.encode_exchange_compose(hb, my, groups_all, n_seg, rank, world, ids, cu, S_in=S_in, via_host=True)
        torch.cuda.synchronize()
        b, e = res.head_begin, res.head_end
        assert (b, e) == ((0, 3) if rank == 0 else (3, 6))
        assert torch.equal(res.E, E0[:, b:e]) and torch.equal(res.T, T0[:, b:e])   # units are independent: bit for bit
        assert torch.equal(res.S, S0[:, b:e])
        assert res.exchanged_bytes == sum(len(g[rank]) for g in groups_all) * (H - (e - b)) * 2 * 128 * 128 * 4
        with open(os.path.join(out_dir, f"ok{rank}"), "w") as f:
            f.write("ok")
    finally:
        dist.destroy_process_group()


def test_two_ranks_one_gpu_shard_exchange_compose_equals_unsharded(tmp_path):
    assert torch.cuda.is_available()
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    assert all((tmp_path / f"ok{r}").exists() for r in range(world))
