"""World-size-2 and -4 gloo tests (CPU) of the multi-GPU orchestration (paper_2008_05612_b200/sharding.py; SURVEY.md
section 8(e)): top-bit shards, rank-local neighbour pass, hypercube exchange for the rank-selecting bits, summed
counts, OR-reduced pair bitmap.  The ranks run the module's own reduce_store_sharded over torch.distributed; the
kernels are stood in for by tests/_cpu_ops.py (no GPU here — tests/test_gpu_sharding.py runs the same module with
libgpmap).  The reduced result must equal the ORACLE's single-rank reductions of the unsharded store."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import gp_oracle as orc
from paper_2008_05612_b200 import sharding
from tests._cpu_ops import NumpyOps


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _store(n_bits, C, seed=7):
    rng = np.random.default_rng(seed)
    ph = rng.integers(0, C, size=1 << n_bits).astype(np.uint16)
    ph = np.sort(ph.reshape(-1, 4), axis=1).reshape(-1)  # some neutral neighbours
    ph[rng.random(1 << n_bits) < 0.6] = 0xFFFF
    return ph


def _worker(rank, world, port, n_bits, C, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ph = _store(n_bits, C)
    b, c = sharding.shard_range(n_bits, world, rank)
    shard = torch.from_numpy(ph[b:b + c].copy().view(np.int16)).view(torch.uint16)
    comm = sharding.DistComm()
    hist, R, D, O, pairs = sharding.reduce_store_sharded(NumpyOps(), comm, shard, n_bits, C, chunk_entries=1000)
    t = comm.max_(1.0 + rank)
    out.put((rank, hist.numpy().copy(), R.numpy().copy(), D.numpy().copy(), O.numpy().copy(), pairs, t, comm.bytes_sent))
    dist.barrier()
    dist.destroy_process_group()


def test_shard_ranges_cover_the_map_and_are_aligned():
    for n_bits, world, align in [(16, 2, 512), (16, 3, 512), (25, 8, 512), (9, 2, 512), (12, 5, 512)]:
        pos = 0
        for r in range(world):
            b, c = sharding.shard_range(n_bits, world, r, align)
            assert b == pos and b % align == 0
            pos = b + c
        assert pos == 1 << n_bits
    with pytest.raises(ValueError):
        sharding.log2_exact(3)
    assert sharding.exchange_bytes_per_rank(36, 8, 28728) == 3 * (2 << 33) + 8 * (4 * 28728 + 1) + 4 * ((28728 ** 2 + 31) // 32)


@pytest.mark.parametrize("world", [2, 4])
def test_sharded_reduction_equals_the_oracle(world):
    n_bits, C = 13, 37
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_bits, C, out)) for r in range(world)]
    for p in procs:
        p.start()
    results = [out.get(timeout=180) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    ph = _store(n_bits, C)
    want_hist = orc.designability(ph, C)
    Ro, Do, Oo, pco = orc.robustness(ph, n_bits, C)
    for rank, hist, R, D, O, pairs, t, sent in results:   # every rank holds the full reduced result
        assert np.array_equal(hist.astype(np.uint64), want_hist), rank
        assert np.array_equal(R.astype(np.uint64), Ro) and np.array_equal(D.astype(np.uint64), Do), rank
        assert np.array_equal(O.astype(np.uint64), Oo) and pairs == pco, rank
        assert t == float(world)
        q = world.bit_length() - 1
        assert sent >= q * 2 * (1 << (n_bits - q))       # at least the shard swaps


def test_single_process_peer_variant_matches_too():
    """PeerComm (all shards in one process, partner shard read in place) + combine_partials: same numbers."""
    n_bits, C, world = 12, 11, 4
    ph = _store(n_bits, C, seed=3)
    shards = []
    for r in range(world):
        b, c = sharding.shard_range(n_bits, world, r)
        shards.append(torch.from_numpy(ph[b:b + c].copy().view(np.int16)).view(torch.uint16))
    ops = NumpyOps()
    parts = [sharding.local_part(ops, sharding.PeerComm(shards, r), shards[r], n_bits, C) for r in range(world)]
    hist, R, D, O, pairs = sharding.combine_partials(ops, parts, C)
    Ro, Do, Oo, pco = orc.robustness(ph, n_bits, C)
    assert np.array_equal(hist.numpy().astype(np.uint64), orc.designability(ph, C))
    assert np.array_equal(R.numpy().astype(np.uint64), Ro) and np.array_equal(D.numpy().astype(np.uint64), Do)
    assert np.array_equal(O.numpy().astype(np.uint64), Oo) and pairs == pco
