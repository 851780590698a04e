"""GPU parity: libgpmap (through the C ABI) against the CPU oracle, bit-exact (integer path: phenotype ids, gaps,
histograms, R/D/O, pair counts, component counts).  Sizes are chosen so the oracle finishes in seconds while the GPU
side still spans several 512-genotype supertiles, several 128-structure tiles, a ragged tail and — for N > 19 —
several prefix batches."""
import numpy as np
import pytest
import torch

import workloads
from oracle import gp_oracle as orc
from paper_2008_05612_b200 import gpmap

pytestmark = pytest.mark.gpu

_lib_structs = {}


def lib_structures(dims):
    if dims not in _lib_structs:
        _lib_structs[dims] = gpmap.Structures(*dims)
    return _lib_structs[dims]


def gpu_enumerate(S, begin, count, simple=False, threshold=1, e=gpmap.HP_ENERGIES, want_gap=True):
    pheno = torch.full((max(count, 1),), 0x1234, dtype=torch.uint16, device="cuda")
    gap = torch.full((max(count, 1),), 77, dtype=torch.int16, device="cuda") if want_gap else None
    S.enumerate(begin, count, pheno, gap, e=e, threshold=threshold, simple=simple)
    torch.cuda.synchronize()
    return pheno[:count].cpu().numpy(), (gap[:count].cpu().numpy() if want_gap else None)


@pytest.mark.parametrize("simple", [False, True])
@pytest.mark.parametrize("dims", [(2, 2, 1), (3, 2, 1), (3, 3, 1), (2, 2, 2), (4, 3, 1), (4, 4, 1)])
def test_full_small_maps(oracle_structures, dims, simple):
    S, O = lib_structures(dims), oracle_structures(*dims)
    total = 1 << S.N
    ph, gap = gpu_enumerate(S, 0, total, simple=simple)
    ph_o, gap_o = O.enumerate(0, total)
    assert np.array_equal(ph, ph_o)
    assert np.array_equal(gap.astype(np.int32), gap_o)


@pytest.mark.parametrize("simple", [False, True])
def test_ranges_5x5(oracle_structures, simple):
    """5x5: ranges inside one prefix batch, across a batch boundary (2^19), and the ragged end of the map."""
    S, O = lib_structures((5, 5, 1)), oracle_structures(5, 5)
    cases = [(0, 3000), ((1 << 19) - 1024, 2048 + 37), ((1 << 25) - 5 * 512, 5 * 512), (13 * (1 << 19) + 512 * 7, 4096)]
    cases += workloads.sample_ranges(25, 4, 2048, 512)[2:]
    for begin, count in cases:
        ph, gap = gpu_enumerate(S, begin, count, simple=simple)
        ph_o, gap_o = O.enumerate(begin, count)
        assert np.array_equal(ph, ph_o), (begin, count)
        assert np.array_equal(gap.astype(np.int32), gap_o), (begin, count)


@pytest.mark.parametrize("fb", [9, 12, 16, 19, 22])
def test_fold_bits_do_not_change_results(oracle_structures, fb):
    """Prefix folding is exact: any split between folded prefix and contraction columns gives the same map."""
    S, O = lib_structures((5, 5, 1)), oracle_structures(5, 5)
    S.tune(fold_bits=fb)
    try:
        for begin, count in [(0, 2048), ((1 << 24) + (1 << fb) - 512, 1536), ((1 << 25) - 2048, 2048)]:
            ph, gap = gpu_enumerate(S, begin, count)
            ph_o, gap_o = O.enumerate(begin, count)
            assert np.array_equal(ph, ph_o), (fb, begin)
            assert np.array_equal(gap.astype(np.int32), gap_o), (fb, begin)
    finally:
        S.tune(fold_bits=15)


@pytest.mark.parametrize("dims,n_ranges,length", [((6, 6, 1), 4, 1024), ((3, 3, 3), 3, 512)])
def test_sampled_ranges_large_lattices(oracle_structures, dims, n_ranges, length):
    """Configs 3 and 4 at full structure count (103 346 / 57 337 columns): sampled genotype ranges vs the oracle."""
    S, O = lib_structures(dims), oracle_structures(*dims)
    for begin, count in workloads.sample_ranges(S.N, n_ranges, length, 512):
        ph, gap = gpu_enumerate(S, begin, count)
        ph_o, gap_o = O.enumerate(begin, count)
        assert np.array_equal(ph, ph_o), (dims, begin)
        assert np.array_equal(gap.astype(np.int32), gap_o), (dims, begin)
        ph_s, _ = gpu_enumerate(S, begin, count, simple=True)
        assert np.array_equal(ph_s, ph_o), (dims, begin)


def test_threshold_and_other_energies(oracle_structures):
    S, O = lib_structures((4, 4, 1)), oracle_structures(4, 4)
    for e, thr in [((0, -10, -10, -23), 4), ((0, -10, -10, -23), 11), ((0, 0, 0, -1), 1), ((-2, -7, -7, -30), 2),
                   ((3, 1, 1, -5), 1)]:
        ph, gap = gpu_enumerate(S, 0, 1 << 16, e=e, threshold=thr)
        ph_o, gap_o = O.enumerate(0, 1 << 16, e=e, threshold=thr)
        assert np.array_equal(ph, ph_o), (e, thr)
        assert np.array_equal(gap.astype(np.int32), gap_o), (e, thr)
        ph_s, gap_s = gpu_enumerate(S, 0, 1 << 16, e=e, threshold=thr, simple=True)
        assert np.array_equal(ph_s, ph_o) and np.array_equal(gap_s.astype(np.int32), gap_o), (e, thr)


def test_edge_cases():
    S = lib_structures((4, 4, 1))
    ph = torch.full((1024,), 0x1234, dtype=torch.uint16, device="cuda")
    S.enumerate(0, 0, ph)  # empty range: nothing written
    S.enumerate(512, 1, ph)  # single genotype
    torch.cuda.synchronize()
    assert int(ph[1]) == 0x1234
    with pytest.raises(gpmap.GpError) as ei:
        S.enumerate(100, 10, ph)
    assert ei.value.status == 5
    with pytest.raises(gpmap.GpError):
        S.enumerate(0, (1 << 16) + 1, torch.empty((1 << 16) + 1, dtype=torch.uint16, device="cuda"))


def test_whole_5x5_map_and_reductions(oracle_structures):
    """Config 2 in full on the GPU: tensor-core path == CUDA-core path; designability, robustness, pair count and
    neutral-network components of the GPU store == the oracle's reductions of the same store; whole-map totals ==
    tests/golden/whole_maps.txt (computed by programs independent of this repository)."""
    from tests._golden import read_whole_maps
    S = lib_structures((5, 5, 1))
    n = 1 << 25
    ph = torch.empty(n, dtype=torch.uint16, device="cuda")
    ph2 = torch.empty(n, dtype=torch.uint16, device="cuda")
    S.enumerate(0, n, ph)
    S.enumerate(0, n, ph2, simple=True)
    assert torch.equal(ph.view(torch.int16), ph2.view(torch.int16))
    hist = gpmap.designability(ph, S.C).cpu().numpy().astype(np.uint64)
    R, Dl, Oc, pc = gpmap.robustness(ph, 25, S.C)
    ncomp = gpmap.nn_components(ph, 25, S.C).cpu().numpy()
    store = ph.cpu().numpy()
    assert np.array_equal(hist, orc.designability(store, S.C))
    Ro, Do, Oo, pco = orc.robustness(store, 25, S.C)
    assert np.array_equal(R.cpu().numpy().astype(np.uint64), Ro)
    assert np.array_equal(Dl.cpu().numpy().astype(np.uint64), Do)
    assert np.array_equal(Oc.cpu().numpy().astype(np.uint64), Oo)
    assert int(pc) == pco
    assert np.array_equal(ncomp.astype(np.uint32), orc.nn_components(store, 25, S.C))
    gold = read_whole_maps()["5x5"]
    assert int(hist[:-1].sum()) == gold["folding"] and int(hist[-1]) == gold["null"]
    assert sorted(hist[:-1].tolist(), reverse=True)[:5] == gold["top5"]
    assert (int(Ro.sum()), int(Do.sum()), int(Oo.sum()), pco) == (gold["sumR"], gold["sumD"], gold["sumO"], gold["pairs"])
    assert int(ncomp.sum()) == gold["nn_total"] and int((ncomp == 1).sum()) == gold["nn_one"] and int(ncomp.max()) == gold["nn_max"]
    # reversal invariance of the map: pheno(rev g) = pheno(g), on a seeded sample
    g = np.random.default_rng(5).integers(0, n, size=200000)
    rev = np.zeros_like(g)
    for i in range(25):
        rev |= ((g >> i) & 1) << (24 - i)
    assert np.array_equal(store[g], store[rev])


@pytest.mark.parametrize("dims", [(3, 3, 1), (4, 4, 1), (2, 2, 2)])
def test_reductions_small(oracle_structures, dims):
    S, O = lib_structures(dims), oracle_structures(*dims)
    n = 1 << S.N
    store = O.enumerate(0, n, want_gap=False)
    ph = torch.from_numpy(store.view(np.int16)).cuda().view(torch.uint16)
    hist = gpmap.designability(ph, S.C).cpu().numpy().astype(np.uint64)
    assert np.array_equal(hist, orc.designability(store, S.C))
    R, Dl, Oc, pc = gpmap.robustness(ph, S.N, S.C)
    Ro, Do, Oo, pco = orc.robustness(store, S.N, S.C)
    assert np.array_equal(R.cpu().numpy().astype(np.uint64), Ro)
    assert np.array_equal(Dl.cpu().numpy().astype(np.uint64), Do)
    assert np.array_equal(Oc.cpu().numpy().astype(np.uint64), Oo)
    assert int(pc) == pco
    ncomp = gpmap.nn_components(ph, S.N, S.C).cpu().numpy()
    assert np.array_equal(ncomp.astype(np.uint32), orc.nn_components(store, S.N, S.C))


def test_reductions_on_synthetic_stores():
    """Reductions are independent of how the store was produced: random stores with a paper-like null fraction,
    ragged histogram lengths, class ids up to the 6x6 count."""
    rng = np.random.default_rng(7)
    for n_bits, C, p_null in [(14, 28728, 0.6), (17, 51704, 0.95), (10, 3, 0.0), (15, 549, 1.0)]:
        n = 1 << n_bits
        store = rng.integers(0, C, size=n).astype(np.uint16)
        store[rng.random(n) < p_null] = 0xFFFF
        ph = torch.from_numpy(store.view(np.int16)).cuda().view(torch.uint16)
        for count in (n, n - 3, 5, 0):
            hist = gpmap.designability(ph[:count] if count else ph[:0], C).cpu().numpy().astype(np.uint64)
            assert np.array_equal(hist, orc.designability(store[:count], C)), (n_bits, count)
        R, Dl, Oc, pc = gpmap.robustness(ph, n_bits, C)
        Ro, Do, Oo, pco = orc.robustness(store, n_bits, C)
        assert np.array_equal(R.cpu().numpy().astype(np.uint64), Ro)
        assert np.array_equal(Dl.cpu().numpy().astype(np.uint64), Do)
        assert np.array_equal(Oc.cpu().numpy().astype(np.uint64), Oo)
        assert int(pc) == pco
        ncomp = gpmap.nn_components(ph, n_bits, C).cpu().numpy()
        assert np.array_equal(ncomp.astype(np.uint32), orc.nn_components(store, n_bits, C))


def test_twenty_letter_variant(oracle_structures):
    """a8 / config 5: seeded sequences + seeded matrix, explicit sequences, and the HP embedding special case."""
    S, O = lib_structures((4, 4, 1)), oracle_structures(4, 4)
    seed = workloads.SEED
    M = gpmap.seeded_matrix(seed)
    count = 50000 + 13
    ph = torch.empty(count, dtype=torch.uint16, device="cuda")
    gap = torch.empty(count, dtype=torch.int16, device="cuda")
    first = (1 << 29) + 77
    S.enumerate_seeded(seed, first, count, ph, gap, e=M)
    seqs = orc.seeded_sequences(seed, first, count, 16)
    ph_o, gap_o = O.enumerate_seqs(seqs, orc.seeded_matrix(seed), 20)
    assert np.array_equal(ph.cpu().numpy(), ph_o)
    assert np.array_equal(gap.cpu().numpy().astype(np.int32), np.maximum(gap_o, -32768))
    # explicit sequences, another matrix, threshold 5
    seqs2 = workloads.random_sequences(20000, 16, 20)
    M2 = workloads.random_symmetric_matrix(20, -300, 40)
    ph2 = torch.empty(20000, dtype=torch.uint16, device="cuda")
    S.enumerate_seqs(torch.from_numpy(seqs2).cuda(), ph2, None, e=M2, alphabet=20, threshold=5)
    assert np.array_equal(ph2.cpu().numpy(), O.enumerate_seqs(seqs2, M2, 20, threshold=5, want_gap=False))
    # HP embedded in 20 letters (letters 0-9 = P, 10-19 = H) reproduces the HP phenotypes
    Mhp = np.zeros((20, 20), np.int32)
    Mhp[10:, :10] = Mhp[:10, 10:] = -10
    Mhp[10:, 10:] = -23
    g = np.arange(1 << 16, dtype=np.uint64)
    bits = ((g[:, None] >> np.arange(16, dtype=np.uint64)[None, :]) & 1).astype(np.uint8)
    letters = (bits * 10 + (g[:, None] % 7).astype(np.uint8)).astype(np.uint8)
    ph3 = torch.empty(1 << 16, dtype=torch.uint16, device="cuda")
    S.enumerate_seqs(torch.from_numpy(letters).cuda(), ph3, None, e=Mhp, alphabet=20)
    assert np.array_equal(ph3.cpu().numpy(), O.enumerate(0, 1 << 16, want_gap=False))


def test_enumerate_host_end_to_end(oracle_structures):
    S, O = lib_structures((4, 4, 1)), oracle_structures(4, 4)
    ph, hist = S.enumerate_host(0, 1 << 16)
    ph_o = O.enumerate(0, 1 << 16, want_gap=False)
    assert np.array_equal(ph, ph_o) and np.array_equal(hist, orc.designability(ph_o, S.C))
    # with the neighbour pass, from a pinned caller buffer
    out = np.empty(1 << 16, np.uint16)
    ph2, hist2, R, Dl, Oc, pc = S.enumerate_host(0, 1 << 16, want_robustness=True, pheno_out=out)
    Ro, Do, Oo, pco = orc.robustness(ph_o, 16, S.C)
    assert ph2 is out and np.array_equal(out, ph_o) and np.array_equal(hist2, hist)
    assert np.array_equal(R, Ro) and np.array_equal(Dl, Do) and np.array_equal(Oc, Oo) and pc == pco
    # a sub-cube of the 5x5 map: flips restricted to the tile's own 12 low bits
    S5, O5 = lib_structures((5, 5, 1)), oracle_structures(5, 5)
    b = 0x1A5 << 12
    ph5, h5, R5, D5, Oc5, pc5 = S5.enumerate_host(b, 1 << 12, want_robustness=True)
    ph5_o = O5.enumerate(b, 1 << 12, want_gap=False)
    Ro, Do, Oo, pco = orc.robustness(ph5_o, 12, S5.C)
    assert np.array_equal(ph5, ph5_o) and np.array_equal(R5, Ro) and np.array_equal(D5, Do) and np.array_equal(Oc5, Oo)
    assert pc5 == pco
    with pytest.raises(gpmap.GpError):
        S5.enumerate_host(512, 1 << 12, want_robustness=True)  # not an aligned sub-cube
    assert gpmap.launch_count() > 0


@pytest.mark.parametrize("tile_bits", [0, 4, 7, 10, 15, 16])
def test_robustness_tile_sizes_agree_with_oracle(tile_bits):
    """The bit-tiled neighbour pass gives the same counts for every tile size (small tiles force the multi-pass,
    spread-bit path on small stores), on stores whose size is not a multiple of the pass width."""
    rng = np.random.default_rng(11)
    for n_bits, C, p_null in [(1, 2, 0.3), (2, 3, 0.3), (3, 5, 0.5), (9, 3, 0.4), (13, 549, 0.6), (18, 28728, 0.57), (21, 51704, 0.95)]:
        n = 1 << n_bits
        store = rng.integers(0, C, size=n).astype(np.uint16)
        # clustered classes, so that neutral neighbours and equal-class runs exist
        store = np.sort(store.reshape(-1, 4), axis=1).reshape(-1) if n >= 4 else store
        store[rng.random(n) < p_null] = 0xFFFF
        ph = torch.from_numpy(store.view(np.int16)).cuda().view(torch.uint16)
        rdo = torch.zeros((3, C), dtype=torch.int64, device="cuda")
        bitmap = gpmap.pair_bitmap(C)
        gpmap.robustness_partial(ph, n_bits, C, rdo, bitmap, tile_bits=tile_bits)
        pc = gpmap.pair_bitmap_count(bitmap, C)
        Ro, Do, Oo, pco = orc.robustness(store, n_bits, C)
        got = rdo.cpu().numpy().astype(np.uint64)
        assert np.array_equal(got[0], Ro), (tile_bits, n_bits)
        assert np.array_equal(got[1], Do), (tile_bits, n_bits)
        assert np.array_equal(got[2], Oo), (tile_bits, n_bits)
        assert int(pc) == pco, (tile_bits, n_bits)
        # without the pair bitmap (other kernel instantiation): same counts
        rdo2 = torch.zeros((3, C), dtype=torch.int64, device="cuda")
        gpmap.robustness_partial(ph, n_bits, C, rdo2, None, tile_bits=tile_bits)
        assert torch.equal(rdo, rdo2), (tile_bits, n_bits)
    # designability and neighbour pass in one sweep (gp_reduce_store) on the last store
    hist, R, Dl, Oc, pc2 = gpmap.reduce_store(ph, n_bits, C)
    assert np.array_equal(hist.cpu().numpy().astype(np.uint64), orc.designability(store, C))
    assert np.array_equal(R.cpu().numpy().astype(np.uint64), Ro) and np.array_equal(Dl.cpu().numpy().astype(np.uint64), Do)
    assert np.array_equal(Oc.cpu().numpy().astype(np.uint64), Oo) and int(pc2) == pco


@pytest.mark.parametrize("C,p_null", [(1, 0.0), (1, 0.5), (2, 0.1), (3, 0.9), (7, 0.36)])
def test_neighbour_pass_on_stores_with_very_few_classes(C, p_null):
    """Stores in which one class holds a large share of the genotypes: the packed per-class words of the direct-table
    kernel wrap thousands of times and every wrap is booked through the carry path; the fused histogram comes from the
    per-call totals.  Default tile size and the small-tile multi-pass path, with and without the pair bitmap."""
    rng = np.random.default_rng(1000 + C)
    n_bits = 20
    n = 1 << n_bits
    store = rng.integers(0, C, size=n).astype(np.uint16)
    store[rng.random(n) < p_null] = 0xFFFF
    Ro, Do, Oo, pco = orc.robustness(store, n_bits, C)
    ph = torch.from_numpy(store.view(np.int16)).cuda().view(torch.uint16)
    for tile_bits in (0, 12):
        rdo = torch.zeros((3, C), dtype=torch.int64, device="cuda")
        bitmap = gpmap.pair_bitmap(C)
        gpmap.robustness_partial(ph, n_bits, C, rdo, bitmap, tile_bits=tile_bits)
        got = rdo.cpu().numpy().astype(np.uint64)
        assert np.array_equal(got[0], Ro) and np.array_equal(got[1], Do) and np.array_equal(got[2], Oo), tile_bits
        assert int(gpmap.pair_bitmap_count(bitmap, C)) == pco
        rdo2 = torch.zeros((3, C), dtype=torch.int64, device="cuda")
        gpmap.robustness_partial(ph, n_bits, C, rdo2, None, tile_bits=tile_bits)
        assert torch.equal(rdo, rdo2), tile_bits
    hist, R, Dl, Oc, pc = gpmap.reduce_store(ph, n_bits, C)
    assert np.array_equal(hist.cpu().numpy().astype(np.uint64), orc.designability(store, C))
    assert np.array_equal(R.cpu().numpy().astype(np.uint64), Ro) and np.array_equal(Dl.cpu().numpy().astype(np.uint64), Do)
    assert np.array_equal(Oc.cpu().numpy().astype(np.uint64), Oo) and int(pc) == pco


@pytest.mark.parametrize("dims,k", [((2, 2, 1), 9), ((3, 3, 1), 9), ((4, 4, 1), 5), ((4, 4, 1), 6), ((4, 4, 1), 8),
                                    ((4, 3, 1), 5), ((4, 3, 1), 7), ((4, 4, 1), 7), ((2, 2, 2), 9)])
def test_enumerate_map_whole_small_maps(oracle_structures, dims, k):
    """gp_enumerate_map (reversal identity, one representative per class) equals the oracle on whole maps, for image
    sizes that give many image pairs, palindromic images and a single image; chains under 10 monomers fall back."""
    S, O = lib_structures(dims), oracle_structures(*dims)
    n = 1 << S.N
    S.tune(sym_bits=k)
    try:
        ph = torch.full((n,), 0x7777, dtype=torch.int32, device="cuda").to(torch.uint16)
        gap = torch.zeros(n, dtype=torch.int16, device="cuda")
        S.enumerate_map(ph, gap)
        torch.cuda.synchronize()
    finally:
        S.tune(sym_bits=7)
    ph_o, gap_o = O.enumerate(0, n)
    assert np.array_equal(ph.cpu().numpy(), ph_o), dims
    assert np.array_equal(gap.cpu().numpy().astype(np.int32), np.maximum(gap_o, -32768)), dims


def test_enumerate_map_other_energies_and_threshold(oracle_structures):
    S, O = lib_structures((4, 4, 1)), oracle_structures(4, 4)
    n = 1 << 16
    S.tune(sym_bits=6)
    try:
        for e, thr in [((0, -10, -10, -23), 4), ((-3, 2, 2, -17), 1), ((5, -1, -1, 0), 2)]:
            ph = torch.empty(n, dtype=torch.uint16, device="cuda")
            S.enumerate_map(ph, None, e=e, threshold=thr)
            assert np.array_equal(ph.cpu().numpy(), O.enumerate(0, n, e=e, threshold=thr, want_gap=False)), (e, thr)
    finally:
        S.tune(sym_bits=7)


def test_bench_step_configuration_sampled(oracle_structures):
    """The step bench.py times (6x6 prefix tile of 2^26 genotypes, gp_enumerate + gp_designability + gp_robustness, same
    launch configuration) checked on sampled outputs the oracle computes one by one, plus the size-independent invariants."""
    import bench
    S, O = lib_structures((6, 6, 1)), oracle_structures(6, 6)
    G, n = 26, 1 << 26
    begin = bench.tile_begin(3, 0, 1, G, S.N)
    ph = torch.empty(n, dtype=torch.uint16, device="cuda")
    S.enumerate(begin, n, ph)
    hist = gpmap.designability(ph, S.C).cpu().numpy().astype(np.int64)
    R, Dl, Oc, pc = (x.cpu().numpy().astype(np.int64) if hasattr(x, "cpu") else x for x in gpmap.robustness(ph, G, S.C))
    assert hist.sum() == n
    folding = int(hist[:S.C].sum())
    assert int(R.sum() + Dl.sum() + Oc.sum()) == G * folding and R.sum() % 2 == 0 and Oc.sum() % 2 == 0
    rng = np.random.default_rng(5)
    offs = np.unique(np.concatenate([[0, n - 1, 511, 512, (1 << 19) - 1, 1 << 19], rng.integers(0, n, 250)]))
    got = ph.view(torch.int16)[torch.from_numpy(offs).cuda()].cpu().numpy().view(np.uint16)
    for o, v in zip(offs.tolist(), got.tolist()):
        assert v == int(O.enumerate(begin + o, 1, want_gap=False)[0]), (begin, o)
    # a whole supertile-aligned stretch as well (ragged against the 2^19 weight-image boundary)
    b2 = (1 << 19) - 256
    assert np.array_equal(ph[b2:b2 + 512].cpu().numpy(), O.enumerate(begin + b2, 512, want_gap=False))


def test_phi_row_against_oracle_transitions(oracle_structures):
    """gp_phi_row(q) equals column q of the oracle's ordered transition matrix (and its null-source entry), on the
    4x4 map, on synthetic stores and on tiny stores."""
    S, O = lib_structures((4, 4, 1)), oracle_structures(4, 4)
    store = O.enumerate(0, 1 << 16, want_gap=False)
    cases = [(store, 16, S.C)]
    rng = np.random.default_rng(3)
    for n_bits, C, p_null in [(1, 2, 0.0), (2, 2, 0.3), (5, 3, 0.4), (13, 40, 0.6)]:
        st = rng.integers(0, C, size=1 << n_bits).astype(np.uint16)
        st[rng.random(1 << n_bits) < p_null] = 0xFFFF
        cases.append((st, n_bits, C))
    for st, n_bits, C in cases:
        T = orc.transitions(st, n_bits, C)
        ph = torch.from_numpy(st.view(np.int16)).cuda().view(torch.uint16)
        n = 1 << n_bits
        idx = np.arange(n, dtype=np.uint64)
        for q in sorted(set([0, C - 1, int(np.argmax(np.bincount(st[st != 0xFFFF], minlength=C)))])):
            row = gpmap.phi_row(ph, n_bits, C, q).cpu().numpy().astype(np.uint64)
            assert np.array_equal(row[:C], T[:, q]), (n_bits, q)
            from_null = sum(int(((st == 0xFFFF) & (st[idx ^ np.uint64(1 << k)] == q)).sum()) for k in range(n_bits))
            assert int(row[C]) == from_null, (n_bits, q)


@pytest.mark.parametrize("dims,count", [((6, 6, 1), 2049), ((3, 3, 3), 1000), ((5, 5, 1), 4096), ((4, 4, 1), 777)])
def test_explicit_hp_sequences_on_tensor_cores(oracle_structures, dims, count):
    """The paper's sampling runs: seeded random H/P sequences, every one against all directed
    structures, through gp_enumerate_seqs (tensor-core sequence_kernel for alphabet 2), against the oracle's explicit
    sequence path, element by element with gaps; ragged counts; then the CUDA-core kernel on a larger batch."""
    import workloads
    S, O = lib_structures(dims), oracle_structures(*dims)
    seqs = workloads.random_sequences(count, S.N, 2)
    seqs[0, :] = 1; seqs[1, :] = 0; seqs[2, :] = np.arange(S.N) % 2          # all-H, all-P, alternating: all null
    e = np.array(gpmap.HP_ENERGIES, np.int32)
    d_seqs = torch.from_numpy(seqs).cuda()
    ph = torch.empty(count, dtype=torch.uint16, device="cuda")
    gap = torch.empty(count, dtype=torch.int16, device="cuda")
    S.enumerate_seqs(d_seqs, ph, gap, e=e, alphabet=2)
    ph_o, gap_o = O.enumerate_seqs(seqs, e, 2)
    assert np.array_equal(ph.cpu().numpy(), ph_o), dims
    assert np.array_equal(gap.cpu().numpy().astype(np.int32), gap_o), dims
    if S.D > 1:
        assert (ph_o[:3] == 0xFFFF).all()
    big = workloads.random_sequences(1 << 15, S.N, 2, seed=11)
    d_big = torch.from_numpy(big).cuda()
    a = torch.empty(1 << 15, dtype=torch.uint16, device="cuda")
    b = torch.empty_like(a)
    S.enumerate_seqs(d_big, a, None, e=e, alphabet=2, threshold=3)
    S.tune(seq_tensor=0)
    try:
        S.enumerate_seqs(d_big, b, None, e=e, alphabet=2, threshold=3)
    finally:
        S.tune(seq_tensor=1)
    assert torch.equal(a.view(torch.int16), b.view(torch.int16)), dims


@pytest.mark.parametrize("dims", [(5, 5, 1), (6, 6, 1)])
def test_letters_outside_the_alphabet_on_every_sequence_kernel(oracle_structures, dims):
    """DESIGN.md reading R19: a byte >= alphabet in an explicit sequence is the last letter.  The three sequence kernels
    (CUDA-core score_simple_kernel, limb seq20_kernel, two-letter sequence_kernel) are picked by gp_tuning.seq_tensor and
    by the batch size (128 and 256 are the switches), so the same bytes go through every setting and through batches on
    both sides of each switch: ids and gaps must equal the oracle's every time."""
    import workloads
    S, O = lib_structures(dims), oracle_structures(*dims)
    rng = np.random.default_rng(1900 + S.N)
    M = orc.seeded_matrix(200805612)
    for alphabet, e, wild in ((2, np.array(gpmap.HP_ENERGIES, np.int32), (2, 3, 7, 128, 255)), (20, M, (20, 21, 64, 200, 255))):
        seqs = workloads.random_sequences(700, S.N, alphabet, seed=19)
        hit = rng.random(seqs.shape) < 0.25
        seqs[hit] = rng.choice(wild, int(hit.sum())).astype(np.uint8)
        seqs[5, :] = 255
        ph_o, gap_o = O.enumerate_seqs(seqs, e, alphabet)
        assert not np.array_equal(ph_o, O.enumerate_seqs(seqs & 1 if alphabet == 2 else seqs % 20, e, alphabet, want_gap=False))
        d_seqs = torch.from_numpy(seqs).cuda()
        try:
            for tensor in (0, 1, 2):
                S.tune(seq_tensor=tensor)
                for count in (100, 200, 300, 700):
                    ph = torch.empty(count, dtype=torch.uint16, device="cuda")
                    gap = torch.empty(count, dtype=torch.int16, device="cuda")
                    S.enumerate_seqs(d_seqs[:count], ph, gap, e=e, alphabet=alphabet)
                    assert np.array_equal(ph.cpu().numpy(), ph_o[:count]), (dims, alphabet, tensor, count)
                    assert np.array_equal(gap.cpu().numpy().astype(np.int32), gap_o[:count]), (dims, alphabet, tensor, count)
        finally:
            S.tune(seq_tensor=1)


@pytest.mark.parametrize("dims,count", [((6, 6, 1), 2500), ((3, 3, 3), 1200), ((4, 4, 1), 700)])
def test_seeded_hp_sequences_drawn_on_chip(oracle_structures, dims, count):
    """The paper's HP sampling runs with the sequences drawn on the GPU (Table 3 HP rows,
    :762-775; the top bit of each draw): gp_enumerate_seeded with alphabet 2 against the oracle on the
    oracle's own copy of the stream — ids and gaps, a first sequence that is not 0, every kernel the call can pick
    (sequence_kernel from 256 sequences on, seq20_kernel from 128, the CUDA-core kernel), a threshold, and other energies."""
    S, O = lib_structures(dims), oracle_structures(*dims)
    seed, first = 200805612, (1 << 33) + 12345
    seqs = orc.seeded_letters(seed, first, count, S.N, 2)
    for e, thr in ((np.array(gpmap.HP_ENERGIES, np.int32), 1), (np.array([1, -7, -7, -19], np.int32), 3)):
        ph_o, gap_o = O.enumerate_seqs(seqs, e, 2, threshold=thr)
        try:
            for tensor in (1, 2, 0):
                S.tune(seq_tensor=tensor)
                for c in (count, 200, 100):
                    ph = torch.empty(c, dtype=torch.uint16, device="cuda")
                    gap = torch.empty(c, dtype=torch.int16, device="cuda")
                    S.enumerate_seeded(seed, first, c, ph, gap, e=e, threshold=thr, alphabet=2)
                    assert np.array_equal(ph.cpu().numpy(), ph_o[:c]), (dims, tensor, c)
                    assert np.array_equal(gap.cpu().numpy().astype(np.int32), gap_o[:c]), (dims, tensor, c)
        finally:
            S.tune(seq_tensor=1)
    # the explicit-sequence call on the library's host copy of the stream gives the same phenotypes
    d_seqs = torch.from_numpy(gpmap.seeded_letters(seed, first, count, S.N, 2)).cuda()
    a = torch.empty(count, dtype=torch.uint16, device="cuda")
    S.enumerate_seqs(d_seqs, a, None, e=np.array(gpmap.HP_ENERGIES, np.int32), alphabet=2)
    assert np.array_equal(a.cpu().numpy(), O.enumerate_seqs(seqs, np.array(gpmap.HP_ENERGIES, np.int32), 2, want_gap=False))
