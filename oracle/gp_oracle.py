"""ctypes binding of the CPU oracle (oracle/gp_oracle.cpp).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It does not
import paper_2008_05612_b200 and shares nothing with it.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gp_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")

NULL_PHENO = 0xFFFF
HP_ENERGIES = (0, -10, -10, -23)  # e[a*2+b], letter 1 = H: E_PP=0, E_HP=-1, E_HH=-2.3, x10


def build(force=False):
    """Compile the oracle with g++ (plain -O2, single-threaded)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".%d.tmp" % os.getpid()
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", _SRC, "-o", tmp])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        vp, u8p, u16p, i32p, u32p, u64p = (ctypes.c_void_p, ctypes.POINTER(ctypes.c_uint8), ctypes.POINTER(ctypes.c_uint16),
                                            ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_uint32),
                                            ctypes.POINTER(ctypes.c_uint64))
        L.oracle_structures_create.restype = vp
        L.oracle_structures_create.argtypes = [ctypes.c_int] * 3
        L.oracle_structures_free.argtypes = [vp]
        for name, rt in (("oracle_length", ctypes.c_int), ("oracle_contacts_per_fold", ctypes.c_int),
                         ("oracle_directed", ctypes.c_uint32), ("oracle_classes", ctypes.c_uint32),
                         ("oracle_self_reverse", ctypes.c_uint32), ("oracle_walk_count", ctypes.c_uint64),
                         ("oracle_group_order", ctypes.c_int)):
            getattr(L, name).restype = rt
            getattr(L, name).argtypes = [vp]
        L.oracle_structure_get.argtypes = [vp, ctypes.c_uint32, u8p, u8p, u32p]
        L.oracle_energy.restype = ctypes.c_int32
        L.oracle_energy.argtypes = [vp, ctypes.c_uint32, u8p, ctypes.c_int, i32p]
        L.oracle_enumerate.argtypes = [vp, i32p, ctypes.c_int32, ctypes.c_uint64, ctypes.c_uint64, u16p, i32p]
        L.oracle_enumerate_seqs.argtypes = [vp, ctypes.c_int, i32p, ctypes.c_int32, u8p, ctypes.c_uint64, u16p, i32p]
        L.oracle_draw.restype = ctypes.c_uint64
        L.oracle_draw.argtypes = [ctypes.c_uint64, ctypes.c_uint64]
        L.oracle_seeded_sequences.argtypes = [ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint64, ctypes.c_int, u8p]
        L.oracle_seeded_letters.argtypes = [ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint64, ctypes.c_int, ctypes.c_int, u8p]
        L.oracle_seeded_matrix.argtypes = [ctypes.c_uint64, i32p]
        L.oracle_designability.argtypes = [u16p, ctypes.c_uint64, ctypes.c_uint32, u64p]
        L.oracle_robustness.argtypes = [u16p, ctypes.c_int, ctypes.c_uint32, u64p, u64p, u64p, u64p]
        L.oracle_transitions.argtypes = [u16p, ctypes.c_int, ctypes.c_uint32, u64p]
        L.oracle_nn_components.argtypes = [u16p, ctypes.c_int, ctypes.c_uint32, u32p]
        _lib = L
    return _lib


def _p(a, ct):
    return a.ctypes.data_as(ctypes.POINTER(ct))


class Structures:
    """Fold library of an nx x ny x nz box, canonicalised per DESIGN.md."""

    def __init__(self, nx, ny, nz=1):
        self._h = lib().oracle_structures_create(nx, ny, nz)
        if not self._h:
            raise ValueError("unsupported lattice %dx%dx%d" % (nx, ny, nz))
        L = lib()
        self.dims = (nx, ny, nz)
        self.N = L.oracle_length(self._h)
        self.NBP = L.oracle_contacts_per_fold(self._h)
        self.D = L.oracle_directed(self._h)
        self.C = L.oracle_classes(self._h)
        self.self_reverse = L.oracle_self_reverse(self._h)
        self.walk_count = L.oracle_walk_count(self._h)
        self.group_order = L.oracle_group_order(self._h)

    def __del__(self):
        if getattr(self, "_h", None):
            lib().oracle_structures_free(self._h)
            self._h = None

    def get(self, d):
        sites = np.zeros(self.N, np.uint8)
        contacts = np.zeros(2 * self.NBP, np.uint8)
        cid = ctypes.c_uint32()
        lib().oracle_structure_get(self._h, d, _p(sites, ctypes.c_uint8), _p(contacts, ctypes.c_uint8), ctypes.byref(cid))
        return sites, contacts.reshape(self.NBP, 2), cid.value

    def tables(self):
        """(sites[D,N], contacts[D,NBP,2], class_of[D]) as numpy arrays."""
        sites = np.zeros((self.D, self.N), np.uint8)
        contacts = np.zeros((self.D, self.NBP, 2), np.uint8)
        class_of = np.zeros(self.D, np.uint32)
        for d in range(self.D):
            s, c, k = self.get(d)
            sites[d], contacts[d], class_of[d] = s, c, k
        return sites, contacts, class_of

    def energy(self, d, letters, e, alphabet=2):
        letters = np.ascontiguousarray(letters, np.uint8)
        e = np.ascontiguousarray(e, np.int32)
        return lib().oracle_energy(self._h, d, _p(letters, ctypes.c_uint8), alphabet, _p(e, ctypes.c_int32))

    def enumerate(self, g_begin, count, e=HP_ENERGIES, threshold=1, want_gap=True):
        e = np.ascontiguousarray(e, np.int32)
        pheno = np.zeros(count, np.uint16)
        gap = np.zeros(count, np.int32) if want_gap else None
        lib().oracle_enumerate(self._h, _p(e, ctypes.c_int32), threshold, g_begin, count, _p(pheno, ctypes.c_uint16),
                               _p(gap, ctypes.c_int32) if want_gap else None)
        return (pheno, gap) if want_gap else pheno

    def enumerate_seqs(self, seqs, e, alphabet, threshold=1, want_gap=True):
        seqs = np.ascontiguousarray(seqs, np.uint8)
        assert seqs.ndim == 2 and seqs.shape[1] == self.N
        e = np.ascontiguousarray(e, np.int32)
        assert e.size == alphabet * alphabet
        count = seqs.shape[0]
        pheno = np.zeros(count, np.uint16)
        gap = np.zeros(count, np.int32) if want_gap else None
        lib().oracle_enumerate_seqs(self._h, alphabet, _p(e, ctypes.c_int32), threshold, _p(seqs, ctypes.c_uint8), count,
                                    _p(pheno, ctypes.c_uint16), _p(gap, ctypes.c_int32) if want_gap else None)
        return (pheno, gap) if want_gap else pheno


def draw(seed, ctr):
    return lib().oracle_draw(seed, ctr)


def seeded_sequences(seed, first, count, N):
    seqs = np.zeros((count, N), np.uint8)
    lib().oracle_seeded_sequences(seed, first, count, N, _p(seqs, ctypes.c_uint8))
    return seqs


def seeded_letters(seed, first, count, N, alphabet):
    """Sequences first..first+count-1 of the DESIGN.md section 4 stream over `alphabet` letters (2 = random H/P)."""
    seqs = np.zeros((count, N), np.uint8)
    lib().oracle_seeded_letters(seed, first, count, N, alphabet, _p(seqs, ctypes.c_uint8))
    return seqs


def seeded_matrix(seed):
    M = np.zeros(400, np.int32)
    lib().oracle_seeded_matrix(seed, _p(M, ctypes.c_int32))
    return M.reshape(20, 20)


def designability(pheno, C):
    pheno = np.ascontiguousarray(pheno, np.uint16)
    hist = np.zeros(C + 1, np.uint64)
    lib().oracle_designability(_p(pheno, ctypes.c_uint16), pheno.size, C, _p(hist, ctypes.c_uint64))
    return hist


def robustness(pheno, n_bits, C):
    """(R, D, O, pair_count) — integer numerators of rho_p, phi_del and the other-phenotype fraction."""
    pheno = np.ascontiguousarray(pheno, np.uint16)
    assert pheno.size == 1 << n_bits
    R, Dl, O = (np.zeros(C, np.uint64) for _ in range(3))
    pc = ctypes.c_uint64()
    lib().oracle_robustness(_p(pheno, ctypes.c_uint16), n_bits, C, _p(R, ctypes.c_uint64), _p(Dl, ctypes.c_uint64),
                            _p(O, ctypes.c_uint64), ctypes.byref(pc))
    return R, Dl, O, pc.value


def transitions(pheno, n_bits, C):
    pheno = np.ascontiguousarray(pheno, np.uint16)
    T = np.zeros((C, C), np.uint64)
    lib().oracle_transitions(_p(pheno, ctypes.c_uint16), n_bits, C, _p(T, ctypes.c_uint64))
    return T


def nn_components(pheno, n_bits, C):
    pheno = np.ascontiguousarray(pheno, np.uint16)
    assert pheno.size == 1 << n_bits
    ncomp = np.zeros(C, np.uint32)
    lib().oracle_nn_components(_p(pheno, ctypes.c_uint16), n_bits, C, _p(ncomp, ctypes.c_uint32))
    return ncomp
