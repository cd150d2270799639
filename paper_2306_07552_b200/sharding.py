"""Multi-GPU host logic: environments are independent, so a batch is sharded
contiguously across ranks, every rank renders its shard with its own scene handle, and there is no collective
on the render path (the paper's layout: 128 environments per GPU x 8 GPUs).  Only timing (max
over ranks) and, if a central consumer wants them, the images are exchanged.  No renderer arithmetic here."""
from __future__ import annotations

from typing import Tuple


def shard_range(n: int, rank: int, world: int) -> Tuple[int, int]:
    """[begin, end) of rank's contiguous shard of n environments; shard sizes differ by at most one."""
    if world <= 0 or not 0 <= rank < world:
        raise ValueError(f"bad rank/world {rank}/{world}")
    q, r = divmod(n, world)
    begin = rank * q + min(rank, r)
    return begin, begin + q + (1 if rank < r else 0)


def max_over_ranks(value: float, device=None) -> float:
    """max of a host scalar over all ranks of the default process group (a no-op without one)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def gather_shards(local, n: int):
    """all-gather equally-typed per-rank arrays (torch tensors, first axis = environments of the shard) into
    the full batch of n environments, in rank order.  For a central consumer; the render path never calls it."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size()
    sizes = [shard_range(n, r, world) for r in range(world)]
    pad = max(e - b for b, e in sizes)
    buf = torch.zeros((pad,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    buf[:local.shape[0]] = local
    out = [torch.empty_like(buf) for _ in range(world)]
    dist.all_gather(out, buf)
    return torch.cat([o[:e - b] for o, (b, e) in zip(out, sizes)], dim=0)


def _rank_main(rank: int, world: int, port: int, target, args) -> None:
    import os
    os.environ.update({"RANK": str(rank), "LOCAL_RANK": str(rank), "WORLD_SIZE": str(world),
                       "MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
    target(*args)


def spawn_ranks(world: int, target, args=()) -> None:
    """Start `world` processes on this node, one per GPU, each with the RANK / LOCAL_RANK / WORLD_SIZE /
    MASTER_* environment torchrun would give it, run target(*args) in every one and wait for all of them
    (what `bench.py --gpus N` does when it was not started under torchrun).  Raises if a rank fails."""
    import socket
    import torch.multiprocessing as mp
    if world < 1:
        raise ValueError("world must be >= 1")
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mp.spawn(_rank_main, args=(world, port, target, tuple(args)), nprocs=world, join=True)
