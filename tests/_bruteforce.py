"""Independent brute force used ONLY to pin the oracle (tests/test_oracle_*.py).

Pure Python on lattice COORDINATES (the oracle works on site indices and contact tables), written from
PAPER.md:65-69 (fold library, Eq. 1) and DESIGN.md's canonical order.  Shares no code with oracle/ or
with the CUDA path.  Only usable on tiny lattices.
"""
import itertools


def hamiltonian_walks(dims):
    """All directed self-avoiding walks visiting every site of the box, as tuples of (x,y,z)."""
    nx, ny, nz = dims
    n = nx * ny * nz
    out = []

    def inside(p):
        return 0 <= p[0] < nx and 0 <= p[1] < ny and 0 <= p[2] < nz

    def extend(walk, used):
        if len(walk) == n:
            out.append(tuple(walk))
            return
        x, y, z = walk[-1]
        for dx, dy, dz in ((1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)):
            p = (x + dx, y + dy, z + dz)
            if inside(p) and p not in used:
                used.add(p)
                walk.append(p)
                extend(walk, used)
                walk.pop()
                used.remove(p)

    for start in itertools.product(range(nx), range(ny), range(nz)):
        extend([start], {start})
    return out


def box_symmetries(dims):
    """Signed axis permutations mapping the box onto itself, as functions on coordinates (deduplicated)."""
    syms = {}
    for perm in itertools.permutations(range(3)):
        if any(dims[perm[a]] != dims[a] for a in range(3)):
            continue
        for flips in itertools.product((False, True), repeat=3):
            def f(p, perm=perm, flips=flips):
                return tuple((dims[a] - 1 - p[perm[a]]) if flips[a] else p[perm[a]] for a in range(3))
            key = tuple(f(p) for p in itertools.product(range(dims[0]), range(dims[1]), range(dims[2])))
            syms.setdefault(key, f)
    return list(syms.values())


def site_index(dims, p):
    return p[0] + dims[0] * (p[1] + dims[1] * p[2])


def classify(dims):
    """Returns (n_walks, directed canonical walks sorted (as site tuples), class_of list, n_self_reverse)."""
    walks = hamiltonian_walks(dims)
    syms = box_symmetries(dims)

    def canon(w):
        return min(tuple(site_index(dims, f(p)) for p in w) for f in syms)

    directed = sorted({canon(w) for w in walks})
    index = {w: d for d, w in enumerate(directed)}
    coords_of = {}
    for w in walks:
        coords_of.setdefault(tuple(site_index(dims, p) for p in w), w)
    rep = []
    self_rev = 0
    for d, w in enumerate(directed):
        dr = index[canon(tuple(reversed(coords_of[w])))]
        self_rev += dr == d
        rep.append(min(d, dr))
    reps = sorted(set(rep))
    class_of = [reps.index(r) for r in rep]
    return len(walks), directed, class_of, self_rev, [coords_of[w] for w in directed]


def contacts_from_coords(walk):
    """Delta of Eq. 1: lattice neighbours that are not chain neighbours."""
    n = len(walk)
    return [(i, j) for i in range(n) for j in range(i + 2, n)
            if sum(abs(a - b) for a, b in zip(walk[i], walk[j])) == 1]


def energy_from_coords(walk, letters, e, alphabet):
    """Eq. 1 evaluated directly on coordinates."""
    return sum(e[letters[i] * alphabet + letters[j]] for i, j in contacts_from_coords(walk))


def ground_state(coords_walks, class_of, letters, e, alphabet, threshold=1):
    """(phenotype or None, m1 - m2 or None) by sorting all energies (a different route from the oracle's scan)."""
    energies = sorted((energy_from_coords(w, letters, e, alphabet), d) for d, w in enumerate(coords_walks))
    if len(energies) == 1:
        return class_of[energies[0][1]], None
    gap = energies[0][0] - energies[1][0]
    return (class_of[energies[0][1]] if -gap >= threshold else None), gap
