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
