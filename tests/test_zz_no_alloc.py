"""gp_threshold_sweep_static — the threshold sweep for callers that cannot allocate device
memory while they run: a service that spent its device-memory budget at start-up, a process whose memory pool is capped
or switched off, a loop where an allocator call is too slow or may synchronise.  The entry point counts in a fixed 4 MiB
device array inside the library instead of asking the stream-ordered pool for a table, so it has a size limit and all
calls share (and must clear) that array.

What is checked, through the C ABI: two calls in a row give exactly the integers gp_threshold_sweep gives (the counts
are integers, so the tolerance of the other sweep tests applies: none), with the second call smaller than the first so
that anything the first call left in the shared array would show; the free device memory does not drop across a call
once the per-device set-up is done; a problem beyond the limit is refused with GP_TOO_LARGE and leaves the outputs alone.

This file sorts last on purpose (pytest -x stops at the first failure; a failure here hides nothing after it) and does
not depend on any other test having run."""
import numpy as np
import pytest
import torch

from paper_2008_05612_b200 import gpmap

pytestmark = pytest.mark.gpu


def _synthetic_store(rng, n, C):
    """(pheno uint16, gap int16) device tensors shaped like a threshold-1 enumeration: mostly null, small gaps, a few
    entries with no second structure."""
    ph = rng.integers(0, C, size=n).astype(np.uint16)
    ph[rng.random(n) < 0.6] = 0xFFFF
    gap = -rng.integers(1, 40, size=n).astype(np.int16)
    gap[rng.random(n) < 0.01] = -32768
    return torch.from_numpy(ph.view(np.int16)).cuda().view(torch.uint16), torch.from_numpy(gap).cuda()


def test_static_sweep_equals_the_allocating_sweep_on_two_calls_in_a_row():
    rng = np.random.default_rng(605612)
    # first call: close to the limit and on the global-atomic path (9 x 51 704 = 465 336 counters of 524 288);
    # second call: few classes, shared-memory path, ragged count — it reuses the low part of the array the first filled
    cases = [((1 << 20) + 77, 51704, [1, 2, 5, 9, 30, 3, 4, 12]), (70001, 40, [7, 1, 4])]
    stores = [_synthetic_store(rng, n, C) for n, C, _ in cases]
    want = [gpmap.threshold_sweep(ph, gap, C, thr) for (ph, gap), (_, C, thr) in zip(stores, cases)]
    outs = [(torch.full((len(thr),), -1, dtype=torch.int64, device="cuda"),
             torch.full((len(thr), C + 1), -1, dtype=torch.int64, device="cuda")) for _, C, thr in cases]
    torch.cuda.synchronize()
    got = []
    for i, ((ph, gap), (_, C, thr)) in enumerate(zip(stores, cases)):
        if i == 1:   # the set-up of this device happened in the first call: from here on nothing may be allocated
            torch.cuda.synchronize()
            free_before = torch.cuda.mem_get_info()[0]
        got.append(gpmap.threshold_sweep_static(ph, gap, C, thr, out=outs[i]))
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before, "the second call took device memory"
    for (f_want, h_want), (f_got, h_got), (n, C, thr) in zip(want, got, cases):
        assert torch.equal(f_got, f_want) and torch.equal(h_got, h_want), (n, C)
        assert int(h_got[0].sum()) == n     # every genotype is either in a class or counted as non-folding
    # a third call with the first input again, after the small one: same answer as before
    f3, h3 = gpmap.threshold_sweep_static(*stores[0], cases[0][1], cases[0][2])
    assert torch.equal(f3, want[0][0]) and torch.equal(h3, want[0][1])
    # an empty store: all zeros (the array is cleared even when no counting kernel runs)
    f0, h0 = gpmap.threshold_sweep_static(stores[1][0][:0], stores[1][1][:0], 40, [1, 5])
    assert int(f0.abs().sum()) == 0 and int(h0.abs().sum()) == 0


def test_static_sweep_on_a_real_map_and_its_size_limit():
    """The whole 4x4 map (enumerated by the library, gaps included) through both sweeps; then a table one class too
    large for the fixed array, which must be refused without touching the outputs."""
    S = gpmap.Structures(4, 4)
    n = 1 << S.N
    ph = torch.empty(n, dtype=torch.uint16, device="cuda")
    gap = torch.empty(n, dtype=torch.int16, device="cuda")
    S.enumerate(0, n, ph, gap)
    thr = [10, 1, 24, 3, 2]
    f_want, h_want = gpmap.threshold_sweep(ph, gap, S.C, thr)
    for _ in range(2):
        f_got, h_got = gpmap.threshold_sweep_static(ph, gap, S.C, thr)
        assert torch.equal(f_got, f_want) and torch.equal(h_got, h_want)
    S.close()
    # 17 x 30 841 = 524 297 > 2^19; 16 x 32 768 = 2^19 exactly is still accepted
    C_big = gpmap.SWEEP_STATIC_MAX_BINS // 17 + 1
    out = (torch.full((16,), -7, dtype=torch.int64, device="cuda"), torch.full((16, C_big + 1), -7, dtype=torch.int64, device="cuda"))
    with pytest.raises(gpmap.GpError) as ei:
        gpmap.threshold_sweep_static(ph, gap, C_big, list(range(1, 17)), out=out)
    assert ei.value.status == 6 and "scratch" in str(ei.value)
    torch.cuda.synchronize()
    assert int((out[0] != -7).sum()) == 0 and int((out[1] != -7).sum()) == 0
    rng = np.random.default_rng(3)
    d_ph, d_gap = _synthetic_store(rng, 4099, 32768)
    thr15 = list(range(1, 16))
    f_want, h_want = gpmap.threshold_sweep(d_ph, d_gap, 32768, thr15)
    f_got, h_got = gpmap.threshold_sweep_static(d_ph, d_gap, 32768, thr15)
    assert torch.equal(f_got, f_want) and torch.equal(h_got, h_want)
