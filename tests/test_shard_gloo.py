"""world_size-2 gloo test (CPU) of the N>1 host logic: member sharding, the one series gather
and the max-over-ranks timing reduction.  No GPU, no kernels."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1911_03386_b200 import shard


def test_member_range_partitions():
    for total in (1, 7, 8, 128, 1024):
        for world in (1, 2, 3, 8):
            blocks = [shard.member_range(total, r, world) for r in range(world)]
            assert blocks[0][0] == 0 and blocks[-1][1] == total
            assert all(a[1] == b[0] for a, b in zip(blocks, blocks[1:]))
            sizes = [hi - lo for lo, hi in blocks]
            assert max(sizes) - min(sizes) <= 1


def _worker(rank, world, port, total):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    lo, hi = shard.member_range(total, rank, world)
    full = torch.arange(3 * total * 4, dtype=torch.float64).reshape(3, total, 4)
    got = shard.gather_series(full[:, lo:hi].contiguous(), total)
    assert torch.equal(got, full)
    t = shard.max_over_ranks(1.0 + rank)
    assert t == float(world)
    dist.barrier()
    dist.destroy_process_group()


def test_gather_series_world2_gloo():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    mp.spawn(_worker, args=(2, port, 7), nprocs=2, join=True)
