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


def _stub_rank(out_dir):
    """What bench.py's ranks do around the render step, with a stub step: read the torchrun-style environment,
    join the process group, reduce a per-rank time with max, pick this rank's environments."""
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from paper_2306_07552_b200.sharding import max_over_ranks
    rank, world, local = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"]), int(os.environ["LOCAL_RANK"])
    assert os.environ["MASTER_ADDR"] == "127.0.0.1" and local == rank
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import bench
        wl = bench.load_workload(0, 2, rank)           # rank r renders environments 2r, 2r+1 of the recipe
        t = max_over_ranks(1.0 + rank)
        with open(os.path.join(out_dir, f"rank{rank}.txt"), "w") as f:
            f.write(f"{world} {t} {' '.join(str(int(i)) for i in wl.env_ids)}")
    finally:
        dist.destroy_process_group()


def test_spawn_ranks_gives_each_rank_its_environment(tmp_path):
    """sharding.spawn_ranks is what `bench.py --gpus N` uses when it is not started by torchrun."""
    from paper_2306_07552_b200.sharding import spawn_ranks
    spawn_ranks(2, _stub_rank, (str(tmp_path),))
    got = [open(os.path.join(str(tmp_path), f"rank{r}.txt")).read().split() for r in range(2)]
    assert got[0] == ["2", "2.0", "0", "1"] and got[1] == ["2", "2.0", "2", "3"]


def test_bench_refuses_more_gpus_than_visible():
    """`bench.py --gpus 2` must not quietly run on fewer devices (no CUDA device at all in the CPU test run)."""
    import subprocess
    import torch
    if torch.cuda.device_count() >= 2:
        pytest.skip("needs a box with fewer than 2 GPUs")
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode != 0 and "--gpus 2" in (r.stderr + r.stdout)
