"""Multi-GPU path with the real library on one device: the whole 5x5 map scored shard by shard
(each emulated rank calls gp_enumerate on its own top-bit range), every rank's share of designability and of the
neighbour pass computed by libgpmap (gp_robustness_partial on the shard, gp_robustness_cross against the partner
shard for the rank-selecting bits), reduced with gp_pair_bitmap_or / sums: exactly the single-rank hist / R / D / O /
pair count, which in turn equal tests/golden/whole_maps.txt.  The ranks run one after the other (no kernel waits on
another rank's kernel)."""
import numpy as np
import pytest
import torch

from paper_2008_05612_b200 import gpmap, sharding
from tests._golden import read_whole_maps

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("world", [2, 4])
def test_sharded_5x5_map_equals_single_rank(world):
    S = gpmap.Structures(5, 5)
    n_bits, C = S.N, S.C
    whole = torch.empty(1 << n_bits, dtype=torch.uint16, device="cuda")
    S.enumerate_map(whole)
    hist1 = gpmap.designability(whole, C)
    R1, D1, O1, pc1 = gpmap.robustness(whole, n_bits, C)
    ops = sharding.LibOps()
    shards = []
    for r in range(world):
        b, c = sharding.shard_range(n_bits, world, r, gpmap.tile())
        sh = torch.empty(c, dtype=torch.uint16, device="cuda")
        S.enumerate(b, c, sh)                                  # rank-local scoring, no communication
        assert torch.equal(sh.view(torch.int16), whole[b:b + c].view(torch.int16))
        shards.append(sh)
    parts = [sharding.local_part(ops, sharding.PeerComm(shards, r), shards[r], n_bits, C, chunk_entries=1 << 22)
             for r in range(world)]
    hist, R, D, O, pairs = sharding.combine_partials(ops, parts, C)
    assert torch.equal(hist, hist1) and torch.equal(R, R1) and torch.equal(D, D1) and torch.equal(O, O1)
    pairs = int(pairs)
    assert pairs == int(pc1)
    gold = read_whole_maps()["5x5"]
    assert (int(R.sum()), int(D.sum()), int(O.sum()), pairs) == (gold["sumR"], gold["sumD"], gold["sumO"], gold["pairs"])
    assert int(hist[:C].sum()) == gold["folding"]
    S.close()


def test_cross_shard_flip_on_synthetic_stores():
    """gp_robustness_cross alone: two halves of a random store = the flip of the top bit."""
    from oracle import gp_oracle as orc
    rng = np.random.default_rng(5)
    n_bits, C = 12, 300
    store = rng.integers(0, C, size=1 << n_bits).astype(np.uint16)
    store = np.sort(store.reshape(-1, 2), axis=1).reshape(-1)
    store[rng.random(1 << n_bits) < 0.5] = 0xFFFF
    ph = torch.from_numpy(store.view(np.int16)).cuda().view(torch.uint16)
    half = 1 << (n_bits - 1)
    rdo = torch.zeros((3, C), dtype=torch.int64, device="cuda")
    bm = gpmap.pair_bitmap(C)
    for a, b in ((ph[:half], ph[half:]), (ph[half:], ph[:half])):
        gpmap.robustness_partial(a, n_bits - 1, C, rdo, bm)
        gpmap.robustness_cross(a, b, C, rdo, bm)
    Ro, Do, Oo, pco = orc.robustness(store, n_bits, C)
    got = rdo.cpu().numpy().astype(np.uint64)
    assert np.array_equal(got[0], Ro) and np.array_equal(got[1], Do) and np.array_equal(got[2], Oo)
    assert int(gpmap.pair_bitmap_count(bm, C)) == pco


@pytest.mark.parametrize("C,hot", [(300, 0.7), (28728, 0.5), (51704, 0.2)])
def test_cross_shard_flip_with_the_shared_memory_class_table(C, hot):
    """gp_robustness_cross on shards long enough for its per-block class table (packed 11 | 11 | 10-bit fields emptied
    through their half marks): a store with a few very hot classes, so that every field passes its half mark many times
    in every block, against the oracle's neighbour pass of the whole store (Eq. 2) — and, on slices
    that start one entry late (scalar loads, ragged count), against the definition written out in numpy."""
    from oracle import gp_oracle as orc
    rng = np.random.default_rng(C)
    n_bits = 22   # 2^21 entries per shard over 148 blocks: the hot classes pass every field's half mark in every block
    n = 1 << n_bits
    store = rng.integers(0, C, size=n).astype(np.uint16)
    pick = rng.random(n) < hot
    store[pick] = rng.integers(0, 3, size=int(pick.sum())).astype(np.uint16)      # classes 0..2 take most entries
    store[rng.random(n) < 0.4] = 0xFFFF
    half = n >> 1
    store[half:][rng.random(half) < 0.5] = 0                                     # many neutral and to-class-0 pairs across the top bit
    ph = torch.from_numpy(store.view(np.int16)).cuda().view(torch.uint16)
    rdo = torch.zeros((3, C), dtype=torch.int64, device="cuda")
    bm = gpmap.pair_bitmap(C)
    for a, b in ((ph[:half], ph[half:]), (ph[half:], ph[:half])):
        gpmap.robustness_partial(a, n_bits - 1, C, rdo, bm)
        gpmap.robustness_cross(a, b, C, rdo, bm)
    Ro, Do, Oo, pco = orc.robustness(store, n_bits, C)
    got = rdo.cpu().numpy().astype(np.uint64)
    assert np.array_equal(got[0], Ro) and np.array_equal(got[1], Do) and np.array_equal(got[2], Oo)
    assert int(gpmap.pair_bitmap_count(bm, C)) == pco
    # misaligned, ragged slices: entry i of `mine` against entry i of `theirs`
    mine, theirs = store[1:half - 2], store[half + 1:n - 2]
    rdo2 = torch.zeros((3, C), dtype=torch.int64, device="cuda")
    gpmap.robustness_cross(ph[1:half - 2], ph[half + 1:n - 2], C, rdo2, None)
    ok = mine != 0xFFFF
    want = [np.bincount(mine[ok & sel], minlength=C) for sel in (theirs == mine, theirs == 0xFFFF, (theirs != mine) & (theirs != 0xFFFF))]
    assert np.array_equal(rdo2.cpu().numpy(), np.stack(want))


def _rank_main(rank, world, port, out):
    """One rank of a two-process run on the same device: libgpmap for every kernel, torch.distributed (gloo, device
    shards staged through the host) for every exchange.  The two processes never wait for each other inside a kernel."""
    import os
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    S = gpmap.Structures(5, 5)
    b, c = sharding.shard_range(S.N, world, rank, gpmap.tile())
    shard = torch.empty(c, dtype=torch.uint16, device="cuda")
    S.enumerate(b, c, shard)
    comm = sharding.DistComm()
    hist, R, D, O, pairs = sharding.reduce_store_sharded(sharding.LibOps(), comm, shard, S.N, S.C, chunk_entries=1 << 22)
    out.put((rank, hist.cpu().numpy(), R.cpu().numpy(), D.cpu().numpy(), O.cpu().numpy(), int(pairs), comm.bytes_sent))
    dist.barrier()
    dist.destroy_process_group()


def test_two_processes_with_libgpmap_over_torch_distributed():
    """reduce_store_sharded end to end: two processes, each scores and reduces its own top-bit shard of the 5x5 map with
    libgpmap and exchanges shards / counts / bitmap through torch.distributed; every rank ends with the golden whole-map
    integers."""
    import socket
    import torch.multiprocessing as mp
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_rank_main, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    results = [out.get(timeout=300) for _ in range(2)]
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    gold = read_whole_maps()["5x5"]
    for rank, hist, R, D, O, pairs, sent in results:
        assert int(hist[:-1].sum()) == gold["folding"] and int(hist[-1]) == gold["null"], rank
        assert (int(R.sum()), int(D.sum()), int(O.sum()), pairs) == (gold["sumR"], gold["sumD"], gold["sumO"], gold["pairs"]), rank
        assert sent >= 2 << 24                              # one shard swap of 2^24 entries
    assert np.array_equal(results[0][1], results[1][1]) and np.array_equal(results[0][2], results[1][2])


def test_full_map_cli_sharded_under_torchrun(tmp_path):
    """`torchrun -m paper_2008_05612_b200.full_map --sharded` with two ranks (gloo between them when the box has one GPU):
    the summary rank 0 writes carries the golden whole-map integers of the 5x5 lattice and passes its own checks."""
    import json
    import os
    import socket
    import subprocess
    import sys
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = str(tmp_path / "map")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), "-m", "paper_2008_05612_b200.full_map", "--lattice", "5x5", "--out", out, "--sharded"]
    r = subprocess.run(cmd, cwd=root, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    with open(os.path.join(out, "summary.json")) as f:
        s = json.load(f)
    gold = read_whole_maps()["5x5"]
    assert s["world"] == 2 and all(s["checks"].values())
    assert (s["folding"], s["null"], s["sum_R"], s["sum_D"], s["sum_O"], s["phenotype_pairs"]) == \
        (gold["folding"], gold["null"], gold["sumR"], gold["sumD"], gold["sumO"], gold["pairs"])
    assert s["bytes_sent_per_rank"] >= 2 << 24
