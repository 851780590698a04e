"""World-size-2 gloo test (CPU) of the multi-GPU host logic: disjoint aligned genotype shards, summed per-class counts,
max-over-ranks timing.  The kernels themselves are single-GPU and covered by the -m gpu tests."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2008_05612_b200 import sharding


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _store(n_bits, C, seed=7):
    rng = np.random.default_rng(seed)
    ph = rng.integers(0, C, size=1 << n_bits).astype(np.uint16)
    ph[rng.random(1 << n_bits) < 0.6] = 0xFFFF
    return ph


def _worker(rank, world, port, n_bits, C, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ph = _store(n_bits, C)
    b, c = sharding.shard_range(n_bits, world, rank, 512)
    mine = ph[b:b + c]
    hist = torch.zeros(C + 1, dtype=torch.int64)
    hist[:C] = torch.from_numpy(np.bincount(mine[mine != 0xFFFF], minlength=C))
    hist[C] = int((mine == 0xFFFF).sum())
    sharding.reduce_counts(hist)
    t = sharding.max_over_ranks(1.0 + rank)
    if rank == 0:
        out.put((hist.numpy().copy(), t))
    dist.destroy_process_group()


def test_shard_ranges_cover_the_map_and_are_aligned():
    for n_bits, world, align in [(16, 2, 512), (16, 3, 512), (25, 8, 512), (9, 2, 512), (12, 5, 512)]:
        pos = 0
        for r in range(world):
            b, c = sharding.shard_range(n_bits, world, r, align)
            assert b == pos and b % align == 0
            pos = b + c
        assert pos == 1 << n_bits
    tiles = [t for r in range(3) for t in sharding.prefix_tiles(10, 6, 3, r)]
    assert sorted(tiles) == [t << 6 for t in range(16)]


def test_world_size_2_counts_add_up():
    n_bits, C, world = 14, 37, 2
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_bits, C, out)) for r in range(world)]
    for p in procs:
        p.start()
    hist, t = out.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    ph = _store(n_bits, C)
    want = np.bincount(ph[ph != 0xFFFF], minlength=C)
    assert np.array_equal(hist[:C], want) and hist[C] == (ph == 0xFFFF).sum() and hist.sum() == 1 << n_bits
    assert t == 2.0
