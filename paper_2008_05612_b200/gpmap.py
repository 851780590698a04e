"""Thin ctypes binding of libgpmap (include/gpmap.h).  Argument marshalling only: every step of the path runs in
the library's CUDA kernels.  PyTorch supplies device memory and streams.  There is no CPU fallback: a missing or
unbuildable library raises at import of the first call.
"""
import ctypes
import os

import numpy as np

from . import build as _build

NULL_PHENO = 0xFFFF
GAP_NONE = -32768
HP_ENERGIES = (0, -10, -10, -23)  # e[a*2+b], letter 1 = H: E_PP, E_HP, E_HP, E_HH x10

_u8p, _u16p, _i16p = (ctypes.POINTER(ctypes.c_uint8), ctypes.POINTER(ctypes.c_uint16), ctypes.POINTER(ctypes.c_int16))
_i32p, _u32p, _u64p = (ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_uint32), ctypes.POINTER(ctypes.c_uint64))
_vp = ctypes.c_void_p


class _Energies(ctypes.Structure):
    _fields_ = [("alphabet", ctypes.c_int32), ("e", _i32p), ("threshold", ctypes.c_int32)]


class _Tuning(ctypes.Structure):
    _fields_ = [("fold_bits", ctypes.c_int32), ("sym_bits", ctypes.c_int32), ("narrow_rows", ctypes.c_int32),
                ("seq_tensor", ctypes.c_int32)]


# name -> (restype, argtypes); must list every symbol include/gpmap.h declares (tests/test_abi.py checks)
SIGNATURES = {
    "gp_structures": (ctypes.c_int, [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.POINTER(_vp)]),
    "gp_structures_free": (None, [_vp]),
    "gp_structures_length": (ctypes.c_int, [_vp]),
    "gp_structures_directed": (ctypes.c_uint32, [_vp]),
    "gp_structures_classes": (ctypes.c_uint32, [_vp]),
    "gp_structures_self_reverse": (ctypes.c_uint32, [_vp]),
    "gp_structures_walks": (ctypes.c_uint64, [_vp]),
    "gp_structures_contacts_per_fold": (ctypes.c_int, [_vp]),
    "gp_structures_features": (ctypes.c_int, [_vp]),
    "gp_structures_get": (ctypes.c_int, [_vp, ctypes.c_uint32, _u8p, _u8p, _u16p]),
    "gp_tuning_get": (ctypes.c_int, [_vp, ctypes.POINTER(_Tuning)]),
    "gp_tuning_set": (ctypes.c_int, [_vp, ctypes.POINTER(_Tuning)]),
    "gp_tile": (ctypes.c_uint64, []),
    "gp_enumerate": (ctypes.c_int, [_vp, ctypes.POINTER(_Energies), ctypes.c_uint64, ctypes.c_uint64, _vp, _vp, _vp]),
    "gp_enumerate_map": (ctypes.c_int, [_vp, ctypes.POINTER(_Energies), _vp, _vp, _vp]),
    "gp_map_units": (ctypes.c_uint64, [_vp]),
    "gp_map_unit": (ctypes.c_int, [_vp, ctypes.c_uint64, _u64p, ctypes.POINTER(ctypes.c_int)]),
    "gp_map_range_genotypes": (ctypes.c_uint64, [_vp, ctypes.c_uint64, ctypes.c_uint64]),
    "gp_enumerate_map_range": (ctypes.c_int, [_vp, ctypes.POINTER(_Energies), ctypes.c_uint64, ctypes.c_uint64, _vp, _vp,
                                              ctypes.c_int, _vp]),
    "gp_enumerate_simple": (ctypes.c_int, [_vp, ctypes.POINTER(_Energies), ctypes.c_uint64, ctypes.c_uint64, _vp, _vp, _vp]),
    "gp_enumerate_seqs": (ctypes.c_int, [_vp, ctypes.POINTER(_Energies), _vp, ctypes.c_uint64, _vp, _vp, _vp]),
    "gp_enumerate_seeded": (ctypes.c_int, [_vp, ctypes.POINTER(_Energies), ctypes.c_uint64, ctypes.c_uint64,
                                           ctypes.c_uint64, _vp, _vp, _vp]),
    "gp_seeded_matrix": (ctypes.c_int, [ctypes.c_uint64, _i32p]),
    "gp_seeded_sequences": (ctypes.c_int, [ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint64, ctypes.c_int, _u8p]),
    "gp_seeded_letters": (ctypes.c_int, [ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint64, ctypes.c_int, ctypes.c_int, _u8p]),
    "gp_designability": (ctypes.c_int, [_vp, ctypes.c_uint64, ctypes.c_uint32, _vp, _vp]),
    "gp_robustness": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_uint32, _vp, _vp, _vp, _vp, _vp]),
    "gp_reduce_store": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_uint32, _vp, _vp, _vp, _vp, _vp, _vp]),
    "gp_pair_bitmap_words": (ctypes.c_uint64, [ctypes.c_uint32]),
    "gp_robustness_partial": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_uint32, _vp, _vp, _vp, _vp, ctypes.c_int, _vp]),
    "gp_robustness_cross": (ctypes.c_int, [_vp, _vp, ctypes.c_uint64, ctypes.c_uint32, _vp, _vp, _vp, _vp, _vp]),
    "gp_pair_bitmap_or": (ctypes.c_int, [_vp, _vp, ctypes.c_uint32, _vp]),
    "gp_pair_bitmap_count": (ctypes.c_int, [_vp, ctypes.c_uint32, _vp, _vp]),
    "gp_threshold_sweep": (ctypes.c_int, [_vp, _vp, ctypes.c_uint64, ctypes.c_uint32, _i32p, ctypes.c_int, _vp, _vp, _vp]),
    "gp_threshold_sweep_static": (ctypes.c_int, [_vp, _vp, ctypes.c_uint64, ctypes.c_uint32, _i32p, ctypes.c_int, _vp, _vp,
                                                 _vp]),
    "gp_phi_row": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_uint32, ctypes.c_uint32, _vp, _vp]),
    "gp_nn_components": (ctypes.c_int, [_vp, ctypes.c_int, ctypes.c_uint32, _vp, _vp]),
    "gp_enumerate_host": (ctypes.c_int, [_vp, ctypes.POINTER(_Energies), ctypes.c_uint64, ctypes.c_uint64, _vp, _u64p,
                                         _u64p, _u64p]),
    "gp_launch_count": (ctypes.c_uint64, []),
    "gp_kernel_timing": (None, [ctypes.c_int]),
    "gp_kernel_time": (ctypes.c_int, [ctypes.c_int, ctypes.POINTER(ctypes.c_double), _u64p]),
    "gp_probe_i8_peak": (ctypes.c_int, [ctypes.c_int, ctypes.c_double, ctypes.POINTER(ctypes.c_double),
                                        ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]),
    "gp_strerror": (ctypes.c_char_p, [ctypes.c_int]),
    "gp_last_cuda_error": (ctypes.c_char_p, []),
}

_lib = None


def lib():
    """Load (building if stale) libgpmap.so.  Raises if it cannot be built or loaded — never falls back."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = ctypes.CDLL(path)
        for name, (res, args) in SIGNATURES.items():
            f = getattr(L, name)
            f.restype = res
            f.argtypes = args
        _lib = L
    return _lib


class GpError(RuntimeError):
    def __init__(self, status, what):
        L = lib()
        msg = "%s: %s" % (what, L.gp_strerror(status).decode())
        if status == 4:
            msg += " [" + L.gp_last_cuda_error().decode() + "]"
        super().__init__(msg)
        self.status = status


def _check(status, what):
    if status != 0:
        raise GpError(status, what)


def _dptr(t, dtype=None):
    """Device pointer of a CUDA torch tensor (None -> NULL)."""
    if t is None:
        return None
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError("expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise ValueError("expected dtype %s, got %s" % (dtype, t.dtype))
    return ctypes.c_void_p(t.data_ptr())


def _stream(stream):
    if stream is None:
        import torch
        return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    return ctypes.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))


def _energies(e, alphabet, threshold):
    arr = np.ascontiguousarray(e, np.int32).reshape(-1)
    if arr.size != alphabet * alphabet:
        raise ValueError("energies must have alphabet^2 entries")
    en = _Energies(alphabet, arr.ctypes.data_as(_i32p), threshold)
    en._keep = arr
    return en


def tile():
    return int(lib().gp_tile())


def launch_count():
    """Kernels launched by libgpmap in this process so far."""
    return int(lib().gp_launch_count())


KERNEL_SCORING, KERNEL_IMAGE, KERNEL_HIST, KERNEL_ROBUSTNESS = range(4)


def kernel_timing(enable):
    lib().gp_kernel_timing(1 if enable else 0)


def kernel_time(which):
    """(total device ms, launches) of one kernel since the last query (needs kernel_timing(True))."""
    ms, n = ctypes.c_double(), ctypes.c_uint64()
    _check(lib().gp_kernel_time(which, ctypes.byref(ms), ctypes.byref(n)), "gp_kernel_time")
    return ms.value, n.value


def probe_i8_peak(k_steps=2, seconds=0.5):
    """gp_probe_i8_peak: (int8 ops/s of the MMA-only stream, SM clocks per MMA, SM MHz it ran at)."""
    ops, clk, mhz = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
    _check(lib().gp_probe_i8_peak(k_steps, seconds, ctypes.byref(ops), ctypes.byref(clk), ctypes.byref(mhz)),
           "gp_probe_i8_peak")
    return ops.value, clk.value, mhz.value


class Structures:
    """gp_structures handle: the fold library of an nx x ny x nz box."""

    def __init__(self, nx, ny, nz=1):
        h = _vp()
        _check(lib().gp_structures(nx, ny, nz, ctypes.byref(h)), "gp_structures(%d,%d,%d)" % (nx, ny, nz))
        self._h = h
        L = lib()
        self.dims = (nx, ny, nz)
        self.N = L.gp_structures_length(h)
        self.D = L.gp_structures_directed(h)
        self.C = L.gp_structures_classes(h)
        self.self_reverse = L.gp_structures_self_reverse(h)
        self.walk_count = L.gp_structures_walks(h)
        self.NBP = L.gp_structures_contacts_per_fold(h)
        self.K = L.gp_structures_features(h)

    def close(self):
        if getattr(self, "_h", None) and lib is not None:   # at interpreter shutdown the module globals are already gone
            lib().gp_structures_free(self._h)
            self._h = None

    __del__ = close

    def tuning(self):
        """gp_tuning_get as a dict."""
        t = _Tuning()
        _check(lib().gp_tuning_get(self._h, ctypes.byref(t)), "gp_tuning_get")
        return {k: getattr(t, k) for k, _ in _Tuning._fields_}

    def tune(self, **kw):
        """gp_tuning_set: change some fields of the handle's gp_tuning (fold_bits, sym_bits, narrow_rows, seq_tensor)."""
        cur = self.tuning()
        for k in kw:
            if k not in cur:
                raise ValueError("unknown tuning field %s" % k)
        cur.update(kw)
        _check(lib().gp_tuning_set(self._h, ctypes.byref(_Tuning(**cur))), "gp_tuning_set")

    def map_units(self):
        return int(lib().gp_map_units(self._h))

    def map_unit(self, unit):
        """(m, k) of a unit of gp_enumerate_map_range: middle-bit value and free monomers per chain end (k = 0: the
        single unit is the whole map)."""
        m, k = ctypes.c_uint64(), ctypes.c_int()
        _check(lib().gp_map_unit(self._h, unit, ctypes.byref(m), ctypes.byref(k)), "gp_map_unit")
        return m.value, k.value

    def get(self, d):
        sites = np.zeros(self.N, np.uint8)
        contacts = np.zeros(2 * self.NBP, np.uint8)
        cid = ctypes.c_uint16()
        _check(lib().gp_structures_get(self._h, d, sites.ctypes.data_as(_u8p), contacts.ctypes.data_as(_u8p),
                                       ctypes.byref(cid)), "gp_structures_get")
        return sites, contacts.reshape(self.NBP, 2), cid.value

    def tables(self):
        sites = np.zeros((self.D, self.N), np.uint8)
        contacts = np.zeros((self.D, self.NBP, 2), np.uint8)
        class_of = np.zeros(self.D, np.uint32)
        for d in range(self.D):
            s, c, k = self.get(d)
            sites[d], contacts[d], class_of[d] = s, c, k
        return sites, contacts, class_of

    # ---- scoring ----
    def enumerate(self, g_begin, g_count, pheno, gap=None, e=HP_ENERGIES, threshold=1, stream=None, simple=False):
        """gp_enumerate / gp_enumerate_simple into caller-owned CUDA tensors (uint16 / int16)."""
        import torch
        en = _energies(e, 2, threshold)
        f = lib().gp_enumerate_simple if simple else lib().gp_enumerate
        if pheno.numel() < g_count or (gap is not None and gap.numel() < g_count):
            raise ValueError("output tensor too small")
        _check(f(self._h, ctypes.byref(en), g_begin, g_count, _dptr(pheno, torch.uint16), _dptr(gap, torch.int16),
                 _stream(stream)), "gp_enumerate")

    def enumerate_map(self, pheno, gap=None, e=HP_ENERGIES, threshold=1, stream=None):
        """gp_enumerate_map: the whole map (2^N entries) through the reversal identity, half the evaluations."""
        import torch
        en = _energies(e, 2, threshold)
        if pheno.numel() != 1 << self.N or (gap is not None and gap.numel() != 1 << self.N):
            raise ValueError("gp_enumerate_map needs 2^N entries")
        _check(lib().gp_enumerate_map(self._h, ctypes.byref(en), _dptr(pheno, torch.uint16), _dptr(gap, torch.int16),
                                      _stream(stream)), "gp_enumerate_map")

    def map_range_genotypes(self, unit_first, unit_count):
        """Genotype integers of a unit range in the order of the compact layout (uint64 numpy array).  Index
        arithmetic of include/gpmap.h only: image m of a unit holds g = (hi << (N-k)) | (m << k) | lo."""
        out = []
        for u in range(unit_first, unit_first + unit_count):
            m, k = self.map_unit(u)
            if k == 0:
                return np.arange(1 << self.N, dtype=np.uint64)
            mid = self.N - 2 * k
            rev = int(format(m, "0%db" % mid)[::-1], 2) if mid else 0
            t = np.arange(1 << (2 * k), dtype=np.uint64)
            for mm in ([m] if rev == m else [m, rev]):
                out.append(((t >> np.uint64(k)) << np.uint64(self.N - k)) | np.uint64(mm << k) | (t & np.uint64((1 << k) - 1)))
        return np.concatenate(out) if out else np.zeros(0, np.uint64)

    def enumerate_map_range(self, unit_first, unit_count, pheno, gap=None, e=HP_ENERGIES, threshold=1, compact=False,
                            stream=None):
        """gp_enumerate_map_range: units [unit_first, unit_first+unit_count) of the map, into the FULL 2^N store or
        (compact=True) into gp_map_range_genotypes entries ordered like map_range_genotypes()."""
        import torch
        en = _energies(e, 2, threshold)
        need = int(lib().gp_map_range_genotypes(self._h, unit_first, unit_count)) if compact else 1 << self.N
        if pheno.numel() < need or (gap is not None and gap.numel() < need) or (not compact and pheno.numel() != need):
            raise ValueError("gp_enumerate_map_range: output holds %d entries, needs %d" % (pheno.numel(), need))
        _check(lib().gp_enumerate_map_range(self._h, ctypes.byref(en), unit_first, unit_count, _dptr(pheno, torch.uint16),
                                            _dptr(gap, torch.int16), 1 if compact else 0, _stream(stream)),
               "gp_enumerate_map_range")

    def enumerate_seqs(self, seqs, pheno, gap=None, e=None, alphabet=20, threshold=1, stream=None):
        import torch
        en = _energies(e, alphabet, threshold)
        if seqs.dim() != 2 or seqs.shape[1] != self.N:
            raise ValueError("seqs must be [count, N] uint8")
        if pheno.numel() < seqs.shape[0] or (gap is not None and gap.numel() < seqs.shape[0]):
            raise ValueError("output tensor too small")
        _check(lib().gp_enumerate_seqs(self._h, ctypes.byref(en), _dptr(seqs, torch.uint8), seqs.shape[0],
                                       _dptr(pheno, torch.uint16), _dptr(gap, torch.int16), _stream(stream)),
               "gp_enumerate_seqs")

    def enumerate_seeded(self, seed, first, count, pheno, gap=None, e=None, threshold=1, stream=None, alphabet=20):
        """gp_enumerate_seeded: sequences first..first+count-1 of the seeded stream over `alphabet` letters, drawn on chip
        (alphabet 2: random H/P sequences, e = the 2x2 energies)."""
        import torch
        en = _energies(e, alphabet, threshold)
        _check(lib().gp_enumerate_seeded(self._h, ctypes.byref(en), seed, first, count, _dptr(pheno, torch.uint16),
                                         _dptr(gap, torch.int16), _stream(stream)), "gp_enumerate_seeded")

    def enumerate_host(self, g_begin, g_count, e=HP_ENERGIES, threshold=1, want_pheno=True, want_robustness=False,
                       pheno_out=None):
        """gp_enumerate_host: host buffers in and out, host<->device copies inside the call.  pheno_out may be a
        caller-owned (e.g. pinned) uint16 numpy array.  Returns (pheno, hist) or (pheno, hist, R, D, O, pair_count)."""
        en = _energies(e, 2, threshold)
        pheno = pheno_out if pheno_out is not None else (np.empty(g_count, np.uint16) if want_pheno else None)
        if pheno is not None and (pheno.dtype != np.uint16 or pheno.size < g_count or not pheno.flags.c_contiguous):
            raise ValueError("pheno_out must be a contiguous uint16 array of at least g_count entries")
        hist = np.zeros(self.C + 1, np.uint64)
        rdo = np.zeros((3, self.C), np.uint64) if want_robustness else None
        pc = ctypes.c_uint64()
        _check(lib().gp_enumerate_host(self._h, ctypes.byref(en), g_begin, g_count,
                                       ctypes.c_void_p(pheno.ctypes.data) if pheno is not None else None,
                                       hist.ctypes.data_as(_u64p),
                                       rdo.ctypes.data_as(_u64p) if want_robustness else None,
                                       ctypes.byref(pc) if want_robustness else None), "gp_enumerate_host")
        if want_robustness:
            return pheno, hist, rdo[0], rdo[1], rdo[2], pc.value
        return pheno, hist


def seeded_matrix(seed):
    M = np.zeros(400, np.int32)
    _check(lib().gp_seeded_matrix(seed, M.ctypes.data_as(_i32p)), "gp_seeded_matrix")
    return M.reshape(20, 20)


def seeded_sequences(seed, first, count, n):
    s = np.zeros((count, n), np.uint8)
    _check(lib().gp_seeded_sequences(seed, first, count, n, s.ctypes.data_as(_u8p)), "gp_seeded_sequences")
    return s


def seeded_letters(seed, first, count, n, alphabet):
    """Host copy of the stream gp_enumerate_seeded draws on chip, over `alphabet` letters (gp_seeded_letters)."""
    s = np.zeros((count, n), np.uint8)
    _check(lib().gp_seeded_letters(seed, first, count, n, alphabet, s.ctypes.data_as(_u8p)), "gp_seeded_letters")
    return s


def designability(pheno, n_classes, hist=None, stream=None):
    import torch
    if hist is None:
        hist = torch.empty(n_classes + 1, dtype=torch.int64, device=pheno.device)
    _check(lib().gp_designability(_dptr(pheno, torch.uint16), pheno.numel(), n_classes, _dptr(hist, torch.int64),
                                  _stream(stream)), "gp_designability")
    return hist


def robustness(pheno, n_bits, n_classes, want_pairs=True, stream=None):
    """(R, D, O, pair_count) device tensors (int64); pair_count is None if not requested."""
    import torch
    if pheno.numel() != 1 << n_bits:
        raise ValueError("gp_robustness needs the full store of 2^n_bits entries")
    out = torch.empty((3, n_classes), dtype=torch.int64, device=pheno.device)
    pc = torch.empty(1, dtype=torch.int64, device=pheno.device) if want_pairs else None
    _check(lib().gp_robustness(_dptr(pheno, torch.uint16), n_bits, n_classes, _dptr(out[0]), _dptr(out[1]), _dptr(out[2]),
                               _dptr(pc), _stream(stream)), "gp_robustness")
    return out[0], out[1], out[2], pc


def reduce_store(pheno, n_bits, n_classes, want_pairs=True, stream=None):
    """gp_reduce_store: (hist, R, D, O, pair_count) — designability and the neighbour pass in one sweep."""
    import torch
    if pheno.numel() != 1 << n_bits:
        raise ValueError("gp_reduce_store needs the full store of 2^n_bits entries")
    hist = torch.empty(n_classes + 1, dtype=torch.int64, device=pheno.device)
    out = torch.empty((3, n_classes), dtype=torch.int64, device=pheno.device)
    pc = torch.empty(1, dtype=torch.int64, device=pheno.device) if want_pairs else None
    _check(lib().gp_reduce_store(_dptr(pheno, torch.uint16), n_bits, n_classes, _dptr(hist), _dptr(out[0]), _dptr(out[1]),
                                 _dptr(out[2]), _dptr(pc), _stream(stream)), "gp_reduce_store")
    return hist, out[0], out[1], out[2], pc


def pair_bitmap(n_classes, device="cuda"):
    """A zeroed pair bitmap (int32[gp_pair_bitmap_words]) for gp_robustness_partial / _cross."""
    import torch
    return torch.zeros(int(lib().gp_pair_bitmap_words(n_classes)), dtype=torch.int32, device=device)


def robustness_partial(pheno, n_bits, n_classes, rdo, bitmap=None, tile_bits=0, stream=None):
    """gp_robustness_partial: ADD the counts of the n_bits local flips of a sub-cube store into rdo (int64[3, C]) and
    OR its connected pairs into bitmap."""
    import torch
    if pheno.numel() != 1 << n_bits:
        raise ValueError("gp_robustness_partial needs a store of 2^n_bits entries")
    _check(lib().gp_robustness_partial(_dptr(pheno, torch.uint16), n_bits, n_classes, _dptr(rdo[0], torch.int64),
                                       _dptr(rdo[1], torch.int64), _dptr(rdo[2], torch.int64), _dptr(bitmap, torch.int32),
                                       tile_bits, _stream(stream)), "gp_robustness_partial")


def robustness_cross(mine, partner, n_classes, rdo, bitmap=None, stream=None):
    """gp_robustness_cross: entries i of `mine` and `partner` differ in one shard-selecting bit; counts go to mine."""
    import torch
    if mine.numel() != partner.numel():
        raise ValueError("shards differ in size")
    _check(lib().gp_robustness_cross(_dptr(mine, torch.uint16), _dptr(partner, torch.uint16), mine.numel(), n_classes,
                                     _dptr(rdo[0], torch.int64), _dptr(rdo[1], torch.int64), _dptr(rdo[2], torch.int64),
                                     _dptr(bitmap, torch.int32), _stream(stream)), "gp_robustness_cross")


def pair_bitmap_or(dst, src, n_classes, stream=None):
    import torch
    _check(lib().gp_pair_bitmap_or(_dptr(dst, torch.int32), _dptr(src, torch.int32), n_classes, _stream(stream)),
           "gp_pair_bitmap_or")


def pair_bitmap_count(bitmap, n_classes, stream=None):
    import torch
    out = torch.empty(1, dtype=torch.int64, device=bitmap.device)
    _check(lib().gp_pair_bitmap_count(_dptr(bitmap, torch.int32), n_classes, _dptr(out, torch.int64), _stream(stream)),
           "gp_pair_bitmap_count")
    return out


def threshold_sweep(pheno, gap, n_classes, thresholds, stream=None):
    """gp_threshold_sweep: (folding int64[T], hist int64[T, C+1]) from the threshold-1 (pheno, gap) stores."""
    import torch
    thr = np.ascontiguousarray(thresholds, np.int32)
    if gap.numel() != pheno.numel():
        raise ValueError("pheno and gap differ in size")
    folding = torch.empty(thr.size, dtype=torch.int64, device=pheno.device)
    hist = torch.empty((thr.size, n_classes + 1), dtype=torch.int64, device=pheno.device)
    _check(lib().gp_threshold_sweep(_dptr(pheno, torch.uint16), _dptr(gap, torch.int16), pheno.numel(), n_classes,
                                    thr.ctypes.data_as(_i32p), thr.size, _dptr(folding), _dptr(hist), _stream(stream)),
           "gp_threshold_sweep")
    return folding, hist


SWEEP_STATIC_MAX_BINS = 1 << 19  # GP_SWEEP_STATIC_MAX_BINS


def threshold_sweep_static(pheno, gap, n_classes, thresholds, stream=None, out=None):
    """gp_threshold_sweep_static: threshold_sweep for callers that must not allocate device memory while running (a
    fixed start-up memory budget, a capped or disabled pool, a loop that cannot take an allocator call).  The library
    counts in a fixed 4 MiB device array of its own, so (len(thresholds) + 1) * n_classes may not exceed
    SWEEP_STATIC_MAX_BINS (GpError with status 6 otherwise), and calls whose GPU work can overlap must not share a
    device.  `out` = (folding int64[T], hist int64[T, C+1]) device tensors the caller allocated beforehand; without it
    this wrapper allocates them through torch, which only the C call itself avoids.  Returns (folding, hist)."""
    import torch
    thr = np.ascontiguousarray(thresholds, np.int32)
    if gap.numel() != pheno.numel():
        raise ValueError("pheno and gap differ in size")
    if out is None:
        out = (torch.empty(thr.size, dtype=torch.int64, device=pheno.device),
               torch.empty((thr.size, n_classes + 1), dtype=torch.int64, device=pheno.device))
    folding, hist = out
    if folding.numel() != thr.size or hist.numel() != thr.size * (n_classes + 1):
        raise ValueError("out tensors do not match the thresholds / classes")
    _check(lib().gp_threshold_sweep_static(_dptr(pheno, torch.uint16), _dptr(gap, torch.int16), pheno.numel(), n_classes,
                                           thr.ctypes.data_as(_i32p), thr.size, _dptr(folding, torch.int64),
                                           _dptr(hist, torch.int64), _stream(stream)),
           "gp_threshold_sweep_static")
    return folding, hist


def phi_row(pheno, n_bits, n_classes, q, stream=None):
    """gp_phi_row: int64[n_classes+1] counts of single mutations leading from each class (last: from null) into q."""
    import torch
    if pheno.numel() != 1 << n_bits:
        raise ValueError("gp_phi_row needs the full store of 2^n_bits entries")
    row = torch.empty(n_classes + 1, dtype=torch.int64, device=pheno.device)
    _check(lib().gp_phi_row(_dptr(pheno, torch.uint16), n_bits, n_classes, q, _dptr(row, torch.int64), _stream(stream)),
           "gp_phi_row")
    return row


def nn_components(pheno, n_bits, n_classes, stream=None):
    import torch
    if pheno.numel() != 1 << n_bits:
        raise ValueError("gp_nn_components needs the full store of 2^n_bits entries")
    ncomp = torch.empty(n_classes, dtype=torch.int32, device=pheno.device)
    _check(lib().gp_nn_components(_dptr(pheno, torch.uint16), n_bits, n_classes, _dptr(ncomp, torch.int32),
                                  _stream(stream)), "gp_nn_components")
    return ncomp
