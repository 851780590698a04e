"""Seeded, synthetic workload descriptions shared by tests/ and bench.py.

Holds none of the method's arithmetic: only which lattice each BASELINE.json config uses and which genotype ranges /
sequence counts are sampled.  Configs 1-4 are the paper's exhaustive workloads themselves (genotypes are the integers
0..2^N-1, nothing to generate); config 5 stands in for the paper's MJ sampling runs with the
counter-based generator of DESIGN.md section 4, which the oracle and the library each implement for themselves.
"""
import numpy as np

SEED = 200805612  # default seed of DESIGN.md section 4

# BASELINE.json configs[0..4]
CONFIGS = {
    "4x4": dict(dims=(4, 4, 1), N=16, D=69, C=38),
    "5x5": dict(dims=(5, 5, 1), N=25, D=1081, C=549),
    "3x3x3": dict(dims=(3, 3, 3), N=27, D=103346, C=51704),
    "6x6": dict(dims=(6, 6, 1), N=36, D=57337, C=28728),
    "mj4x4": dict(dims=(4, 4, 1), N=16, D=69, C=38, alphabet=20, sequences=1 << 30),
}


def sample_ranges(n_bits, n_ranges, length, align, seed=SEED):
    """`n_ranges` genotype ranges [begin, begin+length) in [0, 2^n_bits): the first, the last, one holding the
    palindrome-rich all-ones neighbourhood boundary, the rest seeded-random; begins are multiples of `align`."""
    total = 1 << n_bits
    length = min(length, total)
    rng = np.random.default_rng(seed + n_bits)
    begins = [0, (total - length) // align * align]
    while len(begins) < n_ranges:
        b = int(rng.integers(0, max(1, (total - length) // align + 1))) * align
        if b not in begins:
            begins.append(b)
    return [(b, length) for b in begins[:n_ranges]]


def random_sequences(count, n, alphabet, seed=SEED):
    """Explicit i.i.d. sequences (the paper's SeqRnd path, with a reproducible generator)."""
    return np.random.default_rng(seed).integers(0, alphabet, size=(count, n), dtype=np.uint8)


def random_symmetric_matrix(alphabet, lo, hi, seed=SEED):
    """Symmetric integer matrix, entries uniform in [lo, hi] (a stand-in for a contact-energy table)."""
    rng = np.random.default_rng(seed + 1)
    m = rng.integers(lo, hi + 1, size=(alphabet, alphabet), dtype=np.int32)
    return np.triu(m) + np.triu(m, 1).T
