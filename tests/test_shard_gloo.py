"""N > 1 host logic on CPU: world_size-2 gloo process group.  The data path has no collective
(maps are independent); what is covered is the ownership of map blocks, the seeded inputs each rank draws, and the
max-over-ranks reduction bench.py applies to its device-measured time."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2208_10154_b200 import inputs, shard


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, nmaps, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ks = shard.rank_map_indices(rank, world, nmaps)
        alm = inputs.gaussian_alm(15, ks, 3003)
        # every rank sees every rank's index block and a checksum of its inputs
        blocks = [None] * world
        dist.all_gather_object(blocks, (ks.tolist(), float(np.abs(alm).sum())))
        t = shard.max_over_ranks(10.0 + rank)          # stand-in for a per-rank device time
        if rank == 0:
            out.put((blocks, t))
    finally:
        dist.destroy_process_group()


def test_two_ranks_own_disjoint_blocks_and_reduce_max():
    world, nmaps = 2, 5
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, nmaps, q)) for r in range(world)]
    for p in procs:
        p.start()
    blocks, t = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    allk = sum((b[0] for b in blocks), [])
    assert sorted(allk) == list(range(world * nmaps))            # disjoint and covering
    assert blocks[0][1] != blocks[1][1]                          # different maps -> different inputs
    # the same global map index gives the same input whichever rank draws it
    ref = inputs.gaussian_alm(15, np.array(blocks[1][0]), 3003)
    assert float(np.abs(ref).sum()) == blocks[1][1]
    assert t == 11.0                                             # max over ranks


def test_split_maps_and_identity_without_group():
    assert shard.split_maps(10, 4) == [(0, 3), (3, 3), (6, 2), (8, 2)]
    assert sum(n for _, n in shard.split_maps(1000, 8)) == 1000
    assert shard.max_over_ranks(3.5) == 3.5
    with pytest.raises(ValueError):
        shard.rank_map_indices(2, 2, 4)
