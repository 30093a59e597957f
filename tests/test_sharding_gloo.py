"""Multi-GPU partition exercised with two CPU processes over gloo.

The path shards with no exchange step: rank g of G traces rays g, g + G, g + 2G, ... into its own
buffers.  Here two processes each (1) compute their shard with gp_workloads.shard, (2) trace it with
the ORACLE (no GPU in this container; the selection arithmetic is what is under test, and
ray_begin/ray_count/ray_stride mean the same thing on both sides of the C-ABI), (3) all-gather the
shards over gloo and check that the interleaved union equals the single-process trace record for
record, and that the max-over-ranks timing reduction bench.py uses returns the larger value.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import gp_workloads as W


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, name, out_dir):
    from oracle import oracle as O
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = W.workload(name)
        b, c, s = W.shard(w, rank, world)
        assert (b, s) == (rank, world)
        rec, _ = O.trace(w, b, c, s, n_threads=1)
        # gather the shard sizes, then the records as bytes (shards may differ by one ray)
        sizes = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
        dist.all_gather(sizes, torch.tensor([c], dtype=torch.int64))
        cmax = int(max(t.item() for t in sizes))
        buf = torch.zeros(cmax * rec.dtype.itemsize, dtype=torch.uint8)
        buf[: rec.nbytes] = torch.from_numpy(rec.view(np.uint8).copy())
        parts = [torch.zeros_like(buf) for _ in range(world)]
        dist.all_gather(parts, buf)
        # bench.py's timing reduction: max over ranks
        t = torch.tensor([10.0 + rank], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        assert t.item() == 10.0 + world - 1
        if rank == 0:
            total = W.n_rays(w)
            whole = np.zeros(total, dtype=rec.dtype)
            for g in range(world):
                n_g = int(sizes[g].item())
                whole[g::world] = parts[g].numpy()[: n_g * rec.dtype.itemsize].view(rec.dtype)
            np.save(os.path.join(out_dir, "union.npy"), whole)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("name", ["C1"])
def test_cyclic_shards_reassemble_the_image(tmp_path, name):
    from oracle import oracle as O
    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, name, str(tmp_path)), nprocs=world, join=True)
    union = np.load(tmp_path / "union.npy")
    w = W.workload(name)
    single, _ = O.trace(w)
    assert union.tobytes() == single.tobytes(), "sharded union differs from the single-process trace"


def test_shards_are_disjoint_and_cover_every_ray():
    for name in ("C1", "C2", "C5a"):
        w = W.workload(name)
        total = W.n_rays(w)
        for world in (1, 2, 3, 8):
            seen = 0
            for rank in range(world):
                b, c, s = W.shard(w, rank, world)
                assert b == rank and s == world
                assert b + (c - 1) * s < total <= b + c * s + (world - 1)
                seen += c
            assert seen == total
