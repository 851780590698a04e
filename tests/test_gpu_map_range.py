"""GPU parity of the rangeable map path (gp_map_units / gp_enumerate_map_range, PAPER.md:206-208, :391, :754, :806;
DESIGN.md section 6.6), of concurrent calls on one handle, of energies at the int8 weight bound, of the threshold sweep
(gp_threshold_sweep) and of the 20-letter CUDA-core path off the 4x4 box — all against the
CPU oracle, bit-exact."""
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


def _oracle_at(O, genotypes, **kw):
    """Oracle phenotypes and gaps of scattered genotypes: runs of consecutive integers are enumerated in one call."""
    g = np.asarray(genotypes, dtype=np.uint64)
    ph = np.empty(g.size, np.uint16)
    gap = np.empty(g.size, np.int32)
    i = 0
    while i < g.size:
        j = i + 1
        while j < g.size and g[j] == g[j - 1] + np.uint64(1):
            j += 1
        ph[i:j], gap[i:j] = O.enumerate(int(g[i]), j - i, **kw)
        i = j
    return ph, gap


@pytest.mark.parametrize("dims,k", [((4, 4, 1), 5), ((4, 4, 1), 7), ((5, 5, 1), 7), ((4, 3, 1), 5), ((3, 3, 1), 7)])
def test_map_ranges_in_any_order_fill_the_same_store(oracle_structures, dims, k):
    """Any partition of the units, in any order, on two streams, fills the store gp_enumerate_map fills; the compact
    layout holds the same values in the order gp_map_unit defines; untouched entries stay untouched."""
    S, O = lib_structures(dims), oracle_structures(*dims)
    n = 1 << S.N
    S.tune(sym_bits=k)
    try:
        U = S.map_units()
        assert int(gpmap.lib().gp_map_range_genotypes(S._h, 0, U)) == n
        want = torch.empty(n, dtype=torch.uint16, device="cuda")
        want_gap = torch.empty(n, dtype=torch.int16, device="cuda")
        S.enumerate_map(want, want_gap)
        if S.N <= 16:
            ph_o, gap_o = O.enumerate(0, n)
            assert np.array_equal(want.cpu().numpy(), ph_o) and np.array_equal(want_gap.cpu().numpy().astype(np.int32), gap_o)
        # a seeded partition, shuffled, alternating between two streams
        rng = np.random.default_rng(17 + k)
        cuts = sorted(set([0, U] + rng.integers(0, U + 1, size=min(U, 7)).tolist()))
        pieces = [(cuts[i], cuts[i + 1] - cuts[i]) for i in range(len(cuts) - 1)]
        rng.shuffle(pieces)
        store = torch.full((n,), 0x7777, dtype=torch.int32, device="cuda").to(torch.uint16)
        gap = torch.full((n,), 77, dtype=torch.int16, device="cuda")
        streams = [torch.cuda.Stream(), torch.cuda.Stream()]
        torch.cuda.synchronize()
        for i, (u0, cnt) in enumerate(pieces):
            S.enumerate_map_range(u0, cnt, store, gap, stream=streams[i % 2])
        torch.cuda.synchronize()
        assert torch.equal(store.view(torch.int16), want.view(torch.int16))
        assert torch.equal(gap, want_gap)
        # one piece alone: exactly its genotypes are written; compact layout == gather of the full store
        u0, cnt = pieces[0]
        alone = torch.full((n,), 0x7777, dtype=torch.int32, device="cuda").to(torch.uint16)
        S.enumerate_map_range(u0, cnt, alone)
        g = S.map_range_genotypes(u0, cnt)
        assert g.size == int(gpmap.lib().gp_map_range_genotypes(S._h, u0, cnt)) and np.unique(g).size == g.size
        mask = np.zeros(n, bool)
        mask[g.astype(np.int64)] = True
        got = alone.cpu().numpy()
        assert np.array_equal(got[mask], want.cpu().numpy()[mask]) and (got[~mask] == 0x7777).all()
        cph = torch.empty(g.size, dtype=torch.uint16, device="cuda")
        cgap = torch.empty(g.size, dtype=torch.int16, device="cuda")
        S.enumerate_map_range(u0, cnt, cph, cgap, compact=True)
        assert np.array_equal(cph.cpu().numpy(), want.cpu().numpy()[g.astype(np.int64)])
        assert np.array_equal(cgap.cpu().numpy(), want_gap.cpu().numpy()[g.astype(np.int64)])
        with pytest.raises(gpmap.GpError) as ei:
            S.enumerate_map_range(U, 1, store)
        assert ei.value.status == 5
        S.enumerate_map_range(U, 0, store)  # empty range at the end: nothing to do
    finally:
        S.tune(sym_bits=7)


def test_map_range_slices_of_the_6x6_map(oracle_structures):
    """BASELINE.json configs[3] in the launch configuration the full run uses (k = 7: 2^22 images of 2^14 genotypes,
    28 728 representative columns + combine): three unit slices — first, last (palindromic images), one seeded in the
    middle — in the compact layout; 2 x 2048 genotypes of every slice (the head of image m and of image rev m, plus
    the slice's last image) against the oracle element by element, phenotype and gap."""
    S, O = lib_structures((6, 6, 1)), oracle_structures(6, 6)
    assert S.tuning()["sym_bits"] == 7
    U = S.map_units()
    assert U == (1 << 21) + (1 << 10) and int(gpmap.lib().gp_map_range_genotypes(S._h, 0, U)) == 1 << 36
    n_pair = (1 << 21) - (1 << 10)                       # units with two images; the 2^11 palindromic m follow
    mid_unit = int(np.random.default_rng(workloads.SEED).integers(1000, n_pair - 1000))
    for u0, cnt in [(0, 3), (U - 5, 5), (mid_unit, 4), (n_pair - 2, 4)]:   # the last one straddles pairs | palindromes
        g = S.map_range_genotypes(u0, cnt)
        ph = torch.empty(g.size, dtype=torch.uint16, device="cuda")
        gap = torch.empty(g.size, dtype=torch.int16, device="cuda")
        S.enumerate_map_range(u0, cnt, ph, gap, compact=True)
        torch.cuda.synchronize()
        ph, gap = ph.cpu().numpy(), gap.cpu().numpy().astype(np.int32)
        img = 1 << 14
        pick = np.concatenate([np.arange(0, 2048), np.arange(img, img + 2048), np.arange(g.size - 1024, g.size)])
        # compact order: the local index runs over the 7 low monomers fastest, so 128-genotype runs are consecutive integers
        ph_o, gap_o = _oracle_at(O, g[pick])
        assert np.array_equal(ph[pick], ph_o), (u0, cnt)
        assert np.array_equal(gap[pick], gap_o), (u0, cnt)
        # reversal symmetry inside the slice: pheno(rev g) = pheno(g), and every genotype's reversal is in the slice
        rev = np.zeros_like(g)
        for i in range(36):
            rev |= ((g >> np.uint64(i)) & np.uint64(1)) << np.uint64(35 - i)
        order = np.argsort(g)
        pos = order[np.searchsorted(g[order], rev)]
        assert np.array_equal(g[pos], rev) and np.array_equal(ph[pos], ph)


def test_compact_and_full_store_layouts_agree_on_3x3x3(oracle_structures):
    S, O = lib_structures((3, 3, 3)), oracle_structures(3, 3, 3)
    n = 1 << 27
    U = S.map_units()
    store = torch.full((n,), 0x7777, dtype=torch.int32, device="cuda").to(torch.uint16)
    u0, cnt = U // 3, 9
    S.enumerate_map_range(u0, cnt, store)
    g = S.map_range_genotypes(u0, cnt)
    cph = torch.empty(g.size, dtype=torch.uint16, device="cuda")
    S.enumerate_map_range(u0, cnt, cph, compact=True)
    gi = torch.from_numpy(g.astype(np.int64)).cuda()
    assert torch.equal(store.view(torch.int16)[gi], cph.view(torch.int16))
    assert int((store.view(torch.int16) != 0x7777).sum()) == g.size - int((cph.view(torch.int16) == 0x7777).sum())
    ph_o, _ = _oracle_at(O, g[:1024])
    assert np.array_equal(cph[:1024].cpu().numpy(), ph_o)


def test_concurrent_calls_on_one_handle(oracle_structures):
    """Two gp_enumerate ranges of the 5x5 map run concurrently on two streams of ONE handle (per-call working memory
    comes from the stream-ordered pool), repeatedly; both equal the oracle."""
    S, O = lib_structures((5, 5, 1)), oracle_structures(5, 5)
    ranges = [(7 << 19, 1 << 19), ((21 << 19) + 512 * 3, (1 << 19) + 1024)]   # each spans weight-image boundaries
    outs = [torch.empty(c, dtype=torch.uint16, device="cuda") for _, c in ranges]
    gaps = [torch.empty(c, dtype=torch.int16, device="cuda") for _, c in ranges]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    torch.cuda.synchronize()
    for rep in range(4):
        for i, (b, c) in enumerate(ranges):
            S.enumerate(b, c, outs[i], gaps[i], stream=streams[i])
    torch.cuda.synchronize()
    for i, (b, c) in enumerate(ranges):
        for off in (0, c // 2 - 256, c - 2048):
            ph_o, gap_o = O.enumerate(b + off, 2048)
            assert np.array_equal(outs[i][off:off + 2048].cpu().numpy(), ph_o), (i, off)
            assert np.array_equal(gaps[i][off:off + 2048].cpu().numpy().astype(np.int32), gap_o), (i, off)
    # and against the CUDA-core kernel in full
    for i, (b, c) in enumerate(ranges):
        ref = torch.empty(c, dtype=torch.uint16, device="cuda")
        S.enumerate(b, c, ref, simple=True)
        assert torch.equal(ref.view(torch.int16), outs[i].view(torch.int16))


@pytest.mark.parametrize("dims", [(5, 5, 1), (6, 6, 1)])
def test_energies_at_the_int8_weight_bound(oracle_structures, dims):
    """Energies whose per-monomer weight reaches the int8 bound (3 contacts x |lin + quad| = 126) run exactly on the
    tensor cores, on both paths; energies beyond it are refused (no silent wrap-around of a folded weight)."""
    S, O = lib_structures(dims), oracle_structures(*dims)
    e = (0, -10, -10, -52)   # lin = -10, quad = -32: a free monomer with three H partners in the prefix weighs -126
    n_pref = S.N - 15
    for begin in (((1 << n_pref) - 1) << 15, (0x2AAAAAAAAA & ((1 << n_pref) - 1)) << 15):   # all-H prefix, alternating prefix
        count = 2048
        ph = torch.empty(count, dtype=torch.uint16, device="cuda")
        gap = torch.empty(count, dtype=torch.int16, device="cuda")
        S.enumerate(begin, count, ph, gap, e=e)
        ph_s = torch.empty(count, dtype=torch.uint16, device="cuda")
        S.enumerate(begin, count, ph_s, None, e=e, simple=True)
        ph_o, gap_o = O.enumerate(begin, count, e=e)
        assert np.array_equal(ph.cpu().numpy(), ph_o) and np.array_equal(ph_s.cpu().numpy(), ph_o), (dims, begin)
        assert np.array_equal(gap.cpu().numpy().astype(np.int32), gap_o), (dims, begin)
    g = S.map_range_genotypes(S.map_units() - 1, 1)       # the all-ones palindromic image
    cph = torch.empty(g.size, dtype=torch.uint16, device="cuda")
    S.enumerate_map_range(S.map_units() - 1, 1, cph, e=e, compact=True)
    ph_o, _ = _oracle_at(O, g[-1024:], e=e)
    assert np.array_equal(cph[-1024:].cpu().numpy(), ph_o)
    for bad in [(0, -10, -10, -60), (0, -43, -43, -86), (0, 10, 10, 60)]:
        with pytest.raises(gpmap.GpError) as ei:
            S.enumerate(0, 512, torch.empty(512, dtype=torch.uint16, device="cuda"), e=bad)
        assert ei.value.status == 1, bad


def test_threshold_sweep(oracle_structures):
    """gp_threshold_sweep over the threshold-1 stores == enumerating again with each threshold and taking the
    designability histogram: the oracle on the whole 4x4 map and on a 5x5 range, the library's own thresholded
    enumeration on the whole 5x5 map."""
    thr = [1, 2, 3, 10, 24]
    S, O = lib_structures((4, 4, 1)), oracle_structures(4, 4)
    n = 1 << 16
    ph = torch.empty(n, dtype=torch.uint16, device="cuda")
    gap = torch.empty(n, dtype=torch.int16, device="cuda")
    S.enumerate(0, n, ph, gap)
    order = [10, 1, 24, 3, 2]   # any order
    folding, hist = gpmap.threshold_sweep(ph, gap, S.C, order)
    for row, t in enumerate(order):
        want = orc.designability(O.enumerate(0, n, threshold=t, want_gap=False), S.C)
        assert np.array_equal(hist[row].cpu().numpy().astype(np.uint64), want), t
        assert int(folding[row]) == int(want[:S.C].sum())
    S5, O5 = lib_structures((5, 5, 1)), oracle_structures(5, 5)
    b, c = 0x155 << 16, (1 << 16) - 37
    ph5 = torch.empty(c, dtype=torch.uint16, device="cuda")
    gap5 = torch.empty(c, dtype=torch.int16, device="cuda")
    S5.enumerate(b, c, ph5, gap5)
    folding, hist = gpmap.threshold_sweep(ph5, gap5, S5.C, thr)
    for row, t in enumerate(thr):
        want = orc.designability(O5.enumerate(b, c, threshold=t, want_gap=False), S5.C)
        assert np.array_equal(hist[row].cpu().numpy().astype(np.uint64), want), t
    n5 = 1 << 25
    full = torch.empty(n5, dtype=torch.uint16, device="cuda")
    fgap = torch.empty(n5, dtype=torch.int16, device="cuda")
    S5.enumerate_map(full, fgap)
    folding, hist = gpmap.threshold_sweep(full, fgap, S5.C, thr)
    again = torch.empty(n5, dtype=torch.uint16, device="cuda")
    for row, t in enumerate(thr):
        S5.enumerate_map(again, None, threshold=t)
        want = gpmap.designability(again, S5.C)
        assert torch.equal(hist[row], want), t
        assert int(folding[row]) == n5 - int(want[S5.C])
    # empty input and D = 1 (every genotype folds at every threshold: the gap is "none")
    f0, h0 = gpmap.threshold_sweep(full[:0], fgap[:0], S5.C, [1, 5])
    assert int(f0.sum()) == 0 and int(h0.sum()) == 0
    S2 = lib_structures((2, 2, 1))
    p2 = torch.empty(16, dtype=torch.uint16, device="cuda")
    g2 = torch.empty(16, dtype=torch.int16, device="cuda")
    S2.enumerate(0, 16, p2, g2)
    f2, h2 = gpmap.threshold_sweep(p2, g2, S2.C, [1, 1000])
    assert f2.tolist() == [16, 16] and h2[:, 0].tolist() == [16, 16]


@pytest.mark.parametrize("tensor", [2, 0])
@pytest.mark.parametrize("dims,count", [((6, 6, 1), 2049), ((5, 5, 1), 3000), ((3, 3, 3), 600), ((4, 4, 1), 1000)])
def test_twenty_letter_sequences_on_large_lattices(oracle_structures, dims, count, tensor):
    """a8 / f3 off the 4x4 box (the paper's MJ rows are 6x6 and 3x3x3): seeded 20-letter sequences and
    the seeded matrix, every sequence against all directed structures, ids and gaps against the oracle — on the tensor
    cores (seq20_kernel: two int8 limbs against the 0/-1 contact incidence matrix) and on the CUDA-core kernel; then
    explicit sequences with another matrix (positive entries too) and a threshold; then a matrix whose spread is beyond
    the limbs' int16 range, which must fall back to the CUDA-core kernel and still be exact."""
    S, O = lib_structures(dims), oracle_structures(*dims)
    S.tune(seq_tensor=tensor)
    try:
        seed = workloads.SEED
        M = gpmap.seeded_matrix(seed)
        first = (1 << 33) + 12345
        ph = torch.empty(count, dtype=torch.uint16, device="cuda")
        gap = torch.empty(count, dtype=torch.int16, device="cuda")
        S.enumerate_seeded(seed, first, count, ph, gap, e=M)
        seqs = orc.seeded_sequences(seed, first, count, S.N)
        assert np.array_equal(gpmap.seeded_sequences(seed, first, 64, S.N), seqs[:64])
        ph_o, gap_o = O.enumerate_seqs(seqs, orc.seeded_matrix(seed), 20)
        assert np.array_equal(ph.cpu().numpy(), ph_o), dims
        assert np.array_equal(gap.cpu().numpy().astype(np.int32), np.maximum(gap_o, -32768)), dims
        n2 = count // 2
        seqs2 = workloads.random_sequences(n2, S.N, 20, seed=3)
        seqs2[0, :] = 7                                       # a homopolymer: every structure ties -> null
        M2 = workloads.random_symmetric_matrix(20, -300, 40)
        ph2 = torch.empty(n2, dtype=torch.uint16, device="cuda")
        gap2 = torch.empty(n2, dtype=torch.int16, device="cuda")
        S.enumerate_seqs(torch.from_numpy(seqs2).cuda(), ph2, gap2, e=M2, alphabet=20, threshold=4)
        ph2_o, gap2_o = O.enumerate_seqs(seqs2, M2, 20, threshold=4)
        assert np.array_equal(ph2.cpu().numpy(), ph2_o), dims
        assert np.array_equal(gap2.cpu().numpy().astype(np.int32), np.maximum(gap2_o, -32768)), dims
        if S.D > 1:
            assert ph2_o[0] == 0xFFFF
        # a 7-letter alphabet with a wide spread: (emax - emin) * NBP > 32000, CUDA-core fallback inside the same call
        wide = int(30000 // S.NBP)
        M3 = workloads.random_symmetric_matrix(7, -wide, wide, seed=9)
        if (int(M3.max()) - int(M3.min())) * S.NBP > 32000:
            seqs3 = workloads.random_sequences(300, S.N, 7, seed=4)
            ph3 = torch.empty(300, dtype=torch.uint16, device="cuda")
            S.enumerate_seqs(torch.from_numpy(seqs3).cuda(), ph3, None, e=M3, alphabet=7)
            assert np.array_equal(ph3.cpu().numpy(), O.enumerate_seqs(seqs3, M3, 7, want_gap=False)), dims
    finally:
        S.tune(seq_tensor=1)


def test_twenty_letter_paths_agree_on_a_large_batch():
    """2^17 seeded 20-letter sequences on 6x6: tensor-core and CUDA-core kernels give identical ids and gaps."""
    S = lib_structures((6, 6, 1))
    n = 1 << 17
    M = gpmap.seeded_matrix(workloads.SEED)
    out = []
    for tensor in (1, 0):
        S.tune(seq_tensor=tensor)
        ph = torch.empty(n, dtype=torch.uint16, device="cuda")
        gap = torch.empty(n, dtype=torch.int16, device="cuda")
        S.enumerate_seeded(workloads.SEED, 77, n, ph, gap, e=M)
        out.append((ph, gap))
    S.tune(seq_tensor=1)
    assert torch.equal(out[0][0].view(torch.int16), out[1][0].view(torch.int16)) and torch.equal(out[0][1], out[1][1])


def test_small_explicit_hp_batches_take_the_cuda_core_branch(oracle_structures):
    """gp_enumerate_seqs with fewer than 256 two-letter sequences stays on the CUDA-core kernel: same answers."""
    S, O = lib_structures((5, 5, 1)), oracle_structures(5, 5)
    for count in (1, 100, 255):
        seqs = workloads.random_sequences(count, S.N, 2, seed=count)
        ph = torch.empty(count, dtype=torch.uint16, device="cuda")
        gap = torch.empty(count, dtype=torch.int16, device="cuda")
        S.enumerate_seqs(torch.from_numpy(seqs).cuda(), ph, gap, e=np.array(gpmap.HP_ENERGIES, np.int32), alphabet=2)
        ph_o, gap_o = O.enumerate_seqs(seqs, np.array(gpmap.HP_ENERGIES, np.int32), 2)
        assert np.array_equal(ph.cpu().numpy(), ph_o) and np.array_equal(gap.cpu().numpy().astype(np.int32), gap_o)


@pytest.mark.parametrize("lattice,golden", [("5x5", "5x5")])
def test_full_map_run_survives_an_interruption(oracle_structures, tmp_path, lattice, golden):
    """full_map.run in 16 chunks of units, stopped after 5 chunks as if the job had died, resumed from progress.json and
    the saved store (the paper's long run appended per run): the finished map equals the
    oracle on seeded ranges, every count equals tests/golden/whole_maps.txt, and equals an uninterrupted run."""
    from paper_2008_05612_b200 import full_map
    from tests._golden import read_whole_maps
    out = str(tmp_path / "map")
    assert full_map.run(lattice, out, chunks=16, checkpoint_store=True, stop_after=5) is None
    import json, os
    prog = json.load(open(os.path.join(out, "progress.json")))
    assert prog["chunks_done"] == 5 and prog["store_saved"]
    summary, pheno, S = full_map.run(lattice, out, chunks=16, checkpoint_store=True, resume=True, keep_store=True)
    assert summary["resumed_at_chunk"] == 5 and all(v is True or v == 0 for v in summary["checks"].values())
    O = oracle_structures(*full_map.LATTICES[lattice])
    for b, c in workloads.sample_ranges(S.N, 6, 2048, 512):
        assert np.array_equal(pheno[b:b + c].cpu().numpy(), O.enumerate(b, c, want_gap=False)), b
    gold = read_whole_maps()[golden]
    assert (summary["folding"], summary["null"], summary["top5_designability"]) == (gold["folding"], gold["null"], gold["top5"])
    assert (summary["sum_R"], summary["sum_D"], summary["sum_O"], summary["phenotype_pairs"]) == (
        gold["sumR"], gold["sumD"], gold["sumO"], gold["pairs"])
    once = full_map.run(lattice, str(tmp_path / "once"), chunks=3)
    for key in ("folding", "sum_R", "sum_D", "sum_O", "phenotype_pairs", "top5_designability"):
        assert once[key] == summary[key], key


def test_threshold_sweep_on_synthetic_stores_with_many_classes():
    """The global-atomic path of gp_threshold_sweep (bins do not fit shared memory: 3x3x3-sized class count) and ragged
    counts, against a numpy restatement of the definition (folds iff second_min - min >= threshold)."""
    rng = np.random.default_rng(21)
    for n, C, thr in [((1 << 20) + 77, 51704, [1, 2, 5, 9, 30]), (5000, 28728, [3]), (1 << 16, 40, [7, 1, 4])]:
        ph = rng.integers(0, C, size=n).astype(np.uint16)
        ph[rng.random(n) < 0.6] = 0xFFFF
        gap = -rng.integers(1, 40, size=n).astype(np.int16)
        gap[rng.random(n) < 0.01] = -32768                     # "no second structure": folds at every threshold
        d_ph = torch.from_numpy(ph.view(np.int16)).cuda().view(torch.uint16)
        d_gap = torch.from_numpy(gap).cuda()
        folding, hist = gpmap.threshold_sweep(d_ph, d_gap, C, thr)
        for row, t in enumerate(thr):
            ok = (ph != 0xFFFF) & ((gap == -32768) | (-gap.astype(np.int32) >= t))
            want = np.bincount(ph[ok], minlength=C)
            assert np.array_equal(hist[row, :C].cpu().numpy(), want), (n, t)
            assert int(hist[row, C]) == n - int(ok.sum()) and int(folding[row]) == int(ok.sum()), (n, t)


def test_int8_peak_probe_is_plausible():
    """gp_probe_i8_peak: an M128 x N128 x K32 int8 MMA cannot take fewer than 64 clocks; the measured peak must sit between
    half and all of the nominal 4.5e15 ops/s, and the reported clock between 1 and 2 GHz."""
    for k_steps in (1, 2, 4):
        ops, clk, mhz = gpmap.probe_i8_peak(k_steps, 0.05)
        assert 64.0 <= clk < 80.0, (k_steps, clk)
        assert 2.2e15 < ops < 4.9e15, (k_steps, ops)
        assert 1000.0 < mhz < 2100.0, (k_steps, mhz)
    with pytest.raises(gpmap.GpError):
        gpmap.probe_i8_peak(5, 0.05)


def test_reduce_store_at_the_bench_tile_size(oracle_structures):
    """gp_reduce_store on a WHOLE 2^26-genotype 6x6 prefix tile — the bench step's tile and the geometry the full 6x6 map
    runs its second pass with (direct-table kernel, 2^15 on-chip tiles, 11 spread bits in 32-byte segments) — and on its
    first 2^24 entries (9 spread bits), against the oracle's designability and neighbour pass of the SAME full stores
    (Eq. 2): histogram, neutral / deleterious / other counts of every class and the pair count.  The
    two oracle sweeps (about 50 s and 11 s of single-threaded CPU) run side by side in threads (ctypes drops the GIL).
    gp_designability + gp_robustness, the separate calls, must give the same integers."""
    from concurrent.futures import ThreadPoolExecutor
    S = lib_structures((6, 6, 1))
    G, n = 26, 1 << 26
    ph = torch.empty(n, dtype=torch.uint16, device="cuda")
    S.enumerate(0x2A5 << G, n, ph)
    store = ph.cpu().numpy()
    with ThreadPoolExecutor(2) as pool:
        jobs = {bits: (pool.submit(orc.robustness, store[:1 << bits], bits, S.C),
                       pool.submit(orc.designability, store[:1 << bits], S.C)) for bits in (26, 24)}
        got = {bits: gpmap.reduce_store(ph[:1 << bits], bits, S.C) for bits in (26, 24)}
        hist = gpmap.designability(ph, S.C)
        R, Dl, Oc, pc = gpmap.robustness(ph, G, S.C)
        h2, R2, D2, O2, pc2 = got[26]
        assert torch.equal(hist, h2) and torch.equal(R, R2) and torch.equal(Dl, D2) and torch.equal(Oc, O2) and int(pc) == int(pc2)
        for bits in (24, 26):
            (Ro, Do, Oo, pco), ho = jobs[bits][0].result(), jobs[bits][1].result()
            h3, R3, D3, O3, pc3 = got[bits]
            assert np.array_equal(h3.cpu().numpy().astype(np.uint64), ho), bits
            assert np.array_equal(R3.cpu().numpy().astype(np.uint64), Ro), bits
            assert np.array_equal(D3.cpu().numpy().astype(np.uint64), Do), bits
            assert np.array_equal(O3.cpu().numpy().astype(np.uint64), Oo), bits
            assert int(pc3) == pco and pco > 0, bits
