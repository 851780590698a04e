"""Pins for the oracle's reductions (oracle_designability, oracle_robustness, oracle_transitions,
oracle_nn_components).  PAPER.md:138-147 (designability, neighbourhood, Eq. 2, robustness, phi_del), :19 (NN)."""
import numpy as np
import pytest

from oracle import gp_oracle as orc
from tests._golden import read_3x3_fixture, read_whole_maps

NULL = orc.NULL_PHENO


@pytest.fixture(scope="module")
def maps(oracle_structures):
    out = {}
    for name, dims in (("3x3", (3, 3, 1)), ("4x4", (4, 4, 1)), ("2x2x2", (2, 2, 2))):
        S = oracle_structures(*dims)
        out[name] = (S, S.enumerate(0, 1 << S.N, want_gap=False))
    return out


def numpy_counts(ph, n, C):
    """Vectorised restatement of the neighbour tallies (different route: whole-array XOR gathers + bincount)."""
    g = np.arange(1 << n)
    R, D, O = (np.zeros(C, np.int64) for _ in range(3))
    pairs = set()
    live = ph != NULL
    for k in range(n):
        q = ph[g ^ (1 << k)]
        R += np.bincount(ph[live & (q == ph)], minlength=C)[:C]
        D += np.bincount(ph[live & (q == NULL)], minlength=C)[:C]
        other = live & (q != ph) & (q != NULL)
        O += np.bincount(ph[other], minlength=C)[:C]
        pairs |= set(zip(np.minimum(ph[other], q[other]).tolist(), np.maximum(ph[other], q[other]).tolist()))
    return R, D, O, len(pairs)


@pytest.mark.parametrize("name", ["3x3", "4x4", "2x2x2"])
def test_robustness_equals_numpy_and_invariants(maps, name):
    S, ph = maps[name]
    n, C = S.N, S.C
    R, D, O, pc = orc.robustness(ph, n, C)
    wR, wD, wO, wpc = numpy_counts(ph, n, C)
    assert (R.astype(np.int64) == wR).all() and (D.astype(np.int64) == wD).all() and (O.astype(np.int64) == wO).all()
    assert pc == wpc
    hist = orc.designability(ph, C)
    assert (hist[:C] == np.bincount(ph[ph != NULL], minlength=C)).all() and hist[C] == (ph == NULL).sum()
    assert ((R + D + O) == n * hist[:C]).all()            # every folding genotype has exactly N neighbours
    assert int(R.sum()) % 2 == 0 and int(O.sum()) % 2 == 0
    T = orc.transitions(ph, n, C)
    assert (T == T.T).all()                               # a mutation and its reverse
    assert (np.diag(T) == R).all() and ((T.sum(1) - np.diag(T)) == O).all()
    assert pc == int((np.triu(T, 1) > 0).sum())
    g = np.arange(1 << n)
    nonnull_nb = sum((ph[g ^ (1 << k)] != NULL).astype(np.int64) for k in range(n))
    assert int(D.sum()) == int(nonnull_nb[ph == NULL].sum())


def test_whole_map_values(maps):
    wm = read_whole_maps()
    fx = read_3x3_fixture()
    for name in ("3x3", "4x4"):
        S, ph = maps[name]
        R, D, O, pc = orc.robustness(ph, S.N, S.C)
        assert (int(R.sum()), int(D.sum()), int(O.sum()), pc) == (wm[name]["sumR"], wm[name]["sumD"], wm[name]["sumO"],
                                                                   wm[name]["pairs"])
        if name == "3x3":
            assert (R.tolist(), D.tolist(), O.tolist()) == (fx["R"], fx["D"], fx["O"])
    S, ph = maps["4x4"]
    nc = orc.nn_components(ph, S.N, S.C)
    assert (int(nc.sum()), int((nc == 1).sum()), int(nc.max())) == (wm["4x4"]["nn_total"], wm["4x4"]["nn_one"], wm["4x4"]["nn_max"])


@pytest.mark.parametrize("name", ["3x3", "4x4", "2x2x2"])
def test_components_equal_scipy(maps, name):
    """Library routine as the independent route: scipy connected_components on the explicit hypercube subgraph."""
    from scipy.sparse import coo_matrix
    from scipy.sparse.csgraph import connected_components
    S, ph = maps[name]
    n = S.N
    g = np.arange(1 << n)
    rows, cols = [], []
    for k in range(n):
        nb = g ^ (1 << k)
        keep = (ph != NULL) & (ph[nb] == ph) & (g < nb)
        rows.append(g[keep]); cols.append(nb[keep])
    A = coo_matrix((np.ones(sum(len(r) for r in rows)), (np.concatenate(rows), np.concatenate(cols))), shape=(1 << n, 1 << n))
    _, labels = connected_components(A, directed=False)
    want = np.zeros(S.C, np.int64)
    for c in range(S.C):
        want[c] = len(np.unique(labels[ph == c]))
    assert (orc.nn_components(ph, n, S.C).astype(np.int64) == want).all()


def test_tiny_handmade_store():
    """n_bits = 3 store written by hand: classes 0,1 and null on the cube's corners."""
    ph = np.array([0, 0, 1, NULL, 0, NULL, 1, 1], np.uint16)   # g = 0..7
    # g=0 (class 0): nb 1->0 R, 2->1 O, 4->0 R ; g=1: nb 0->0 R, 3->null D, 5->null D ; g=4: nb 5->null D, 6->1 O, 0->0 R
    # g=2 (class 1): nb 3->null D, 0->0 O, 6->1 R ; g=6: nb 7->1 R, 4->0 O, 2->1 R ; g=7: nb 6->1 R, 5->null D, 3->null D
    R, D, O, pc = orc.robustness(ph, 3, 2)
    assert (R.tolist(), D.tolist(), O.tolist(), pc) == ([4, 4], [3, 3], [2, 2], 1)
    assert orc.designability(ph, 2).tolist() == [3, 3, 2]
    assert orc.nn_components(ph, 3, 2).tolist() == [1, 1]
    ph2 = np.array([0, NULL, NULL, 0, NULL, 0, 0, NULL], np.uint16)   # even-parity corners: four isolated genotypes
    assert orc.nn_components(ph2, 3, 1).tolist() == [4]
    R, D, O, pc = orc.robustness(ph2, 3, 1)
    assert (R.tolist(), D.tolist(), O.tolist(), pc) == ([0], [12], [0], 0)
