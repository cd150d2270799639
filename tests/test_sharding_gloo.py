"""Multi-process host logic on CPU (gloo, world_size 2): contiguous sharding of a batch, per-rank rendering of
the shard, gather in rank order == the single-process result, and the max-over-ranks timing reduction.  The
renderer on each rank is the CPU oracle here (the GPU path is covered by test_sharding_and_determinism)."""
from __future__ import annotations

import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_shard_range_partitions():
    from paper_2306_07552_b200.sharding import shard_range
    for n in (0, 1, 7, 1024, 1025):
        for world in (1, 2, 3, 8):
            r = [shard_range(n, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(r, r[1:]))
            sizes = [e - b for b, e in r]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_range(4, 2, 2)


def _worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        from paper_2306_07552_b200 import gen
        from paper_2306_07552_b200.sharding import gather_shards, max_over_ranks, shard_range
        wl = gen.make_config(0, n_envs=3)          # 3 environments over 2 ranks: shards of 2 and 1
        b, e = shard_range(wl.N, rank, world)
        o = oracle.render(wl.subset(np.arange(b, e)), n_threads=1)
        depth = gather_shards(torch.from_numpy(o["depth"]), wl.N)
        ids = gather_shards(torch.from_numpy(o["id"].view(np.int32)), wl.N)
        rgb = gather_shards(torch.from_numpy(o["rgb"]), wl.N)
        t = max_over_ranks(10.0 + rank)
        if rank == 0:
            np.savez(os.path.join(out_dir, "gathered.npz"), depth=depth.numpy(), id=ids.numpy().view(np.uint32),
                     rgb=rgb.numpy(), t=t)
    finally:
        dist.destroy_process_group()


def test_two_rank_sharded_render_matches_single(tmp_path, oracle_mod):
    import socket
    import torch.multiprocessing as mp
    from paper_2306_07552_b200 import gen
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    got = np.load(os.path.join(str(tmp_path), "gathered.npz"))
    ref = oracle_mod.render(gen.make_config(0, n_envs=3))
    assert np.array_equal(got["depth"].view(np.uint32), ref["depth"].view(np.uint32))
    assert np.array_equal(got["id"], ref["id"])
    assert np.array_equal(got["rgb"], ref["rgb"])
    assert float(got["t"]) == 11.0
