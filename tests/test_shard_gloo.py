"""N>1 host logic on CPU (gloo, world_size 2): request sharding is a partition with no data-path
collective, and the max-over-ranks timing reduction bench.py uses."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, ret):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    import d2sd_synth as synth
    import oracle
    cfg = synth.custom(95, B=5, gamma=8, K=3, V=64, ctx=(3, 40), Hq=4, Hkv=2)
    st = synth.make_step_inputs(cfg)
    lo, hi = bench.shard_range(cfg.B, rank, world)
    pl, _ = oracle.select_prefixes(st["conf"][lo:hi], cfg.K)
    tree = oracle.build_tree(st["draft1"][lo:hi], st["draft2"][lo:hi], pl, st["ctx_len"][lo:hi], cfg.T_cap)
    # every rank processes only its own requests; results are merely concatenated (no reduction)
    mine = torch.from_numpy(np.concatenate([tree["tree_len"], np.full(cfg.B - (hi - lo), -1, np.int32)]))
    gathered = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(gathered, mine)
    t = bench.max_over_ranks(1.0 + rank)  # rank 1 is slower
    units = bench.sum_over_ranks(float(tree["tree_len"].sum()))
    if rank == 0:
        pl_all, _ = oracle.select_prefixes(st["conf"], cfg.K)
        full = oracle.build_tree(st["draft1"], st["draft2"], pl_all, st["ctx_len"], cfg.T_cap)
        got = np.concatenate([g.numpy()[g.numpy() >= 0] for g in gathered])
        ret["ok"] = bool(np.array_equal(got, full["tree_len"])) and t == 2.0 and units == float(full["tree_len"].sum())
    dist.destroy_process_group()


def test_shard_range_is_a_partition():
    sys.path.insert(0, ROOT)
    import bench
    for B in (0, 1, 5, 16, 17):
        for world in (1, 2, 3, 8):
            spans = [bench.shard_range(B, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == B
            assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
            sizes = [hi - lo for lo, hi in spans]
            assert max(sizes) - min(sizes) <= 1


def test_two_rank_sharding_gloo():
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(2, _free_port(), ret), nprocs=2, join=True)
    assert ret.get("ok") is True
