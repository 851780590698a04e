"""Pins for the oracle's fold library (oracle_structures_*): brute force on coordinates, paper-printed counts,
closed forms.  PAPER.md:65 (library = all compact self-avoiding walks), :454 (57337), :216 (51704)."""
import numpy as np
import pytest

from tests._golden import read_3x3_fixture, read_pins
from tests import _bruteforce as bf

EDGES = lambda d: sum((d[a] - 1) * d[(a + 1) % 3] * d[(a + 2) % 3] for a in range(3))


@pytest.mark.parametrize("dims", [(2, 2, 1), (3, 2, 1), (3, 3, 1), (2, 2, 2), (4, 4, 1), (4, 3, 1)])
def test_library_equals_bruteforce(oracle_structures, dims):
    S = oracle_structures(*dims)
    n_walks, directed, class_of, self_rev, coords = bf.classify(dims)
    assert S.walk_count == n_walks
    assert (S.D, S.C, S.self_reverse) == (len(directed), max(class_of) + 1, self_rev)
    sites, contacts, cls = S.tables()
    assert [tuple(r) for r in sites.tolist()] == directed          # same canonical forms, same order
    assert cls.tolist() == class_of
    for d in range(S.D):
        assert [tuple(c) for c in contacts[d].tolist()] == bf.contacts_from_coords(coords[d])


def test_3x3_permutation_count():
    """Route independent of any DFS: count permutations of the 9 sites whose consecutive sites are adjacent."""
    import itertools
    adj = lambda a, b: abs(a % 3 - b % 3) + abs(a // 3 - b // 3) == 1
    n = sum(all(adj(p[i], p[i + 1]) for i in range(8)) for p in itertools.permutations(range(9)))
    assert n == 40


def test_3x3_fixture(oracle_structures):
    S = oracle_structures(3, 3)
    fx = read_3x3_fixture()
    assert S.D == len(fx["structures"])
    for s in fx["structures"]:
        sites, contacts, cls = S.get(s["d"])
        assert sites.tolist() == s["sites"] and cls == s["cls"]
        assert [tuple(c) for c in contacts.tolist()] == s["contacts"]


@pytest.mark.parametrize("dims,group", [((2, 2, 1), 8), ((3, 3, 1), 8), ((4, 4, 1), 8), ((5, 5, 1), 8), ((6, 6, 1), 8),
                                        ((2, 2, 2), 48), ((3, 3, 3), 48), ((3, 2, 1), 4)])
def test_closed_forms(oracle_structures, dims, group):
    S = oracle_structures(*dims)
    assert S.group_order == group
    # a compact directed walk has trivial stabiliser => D = walks / |G| exactly; C = (D + self-reverse) / 2
    assert S.walk_count == S.D * group
    assert 2 * S.C == S.D + S.self_reverse
    assert S.NBP == EDGES(dims) - (S.N - 1)
    sites, contacts, cls = S.tables()
    assert all(sorted(r) == list(range(S.N)) for r in sites[:: max(1, S.D // 200)].tolist())
    i, j = contacts[..., 0].astype(int), contacts[..., 1].astype(int)
    assert ((j - i) % 2 == 1).all() and ((j - i) >= 3).all()       # bipartite lattice
    first = np.unique(cls, return_index=True)[1]                  # class ids are ranked by their smallest member
    assert (np.diff(first) > 0).all() and cls[0] == 0 and cls.max() == S.C - 1
    order = np.lexsort(sites.T[::-1])
    assert (order == np.arange(S.D)).all()                        # lexicographic order of canonical forms


def test_paper_counts(oracle_structures):
    pins = read_pins()
    s66, s333 = oracle_structures(6, 6), oracle_structures(3, 3, 3)
    assert s66.D == pins["folds_6x6_directed"] and s66.N == pins["length_6x6"]
    assert s333.C == pins["folds_3x3x3_classes"]
    assert s333.D == 103346 and s333.D == 2 * s333.C - s333.self_reverse           # DESIGN.md reading R2
    assert (s66.C, s66.self_reverse, s66.NBP, s333.NBP) == (28728, 119, 25, 28)
    assert (oracle_structures(5, 5).D, oracle_structures(5, 5).C) == (1081, 549)
