"""CPU-side checks of the C-ABI library: it builds for sm_100a, loads, exports every symbol include/gpmap.h declares,
rejects bad arguments, and its host-side gp_structures (a0) agrees with the oracle's fold library table by table.
No compute calls (no GPU here)."""
import ctypes
import os
import re

import numpy as np
import pytest

from oracle import gp_oracle as orc
from paper_2008_05612_b200 import build as gbuild
from paper_2008_05612_b200 import gpmap
from tests._golden import read_pins

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_builds_and_exports_every_declared_symbol():
    path = gbuild.build()
    assert os.path.exists(path)
    L = ctypes.CDLL(path)
    header = open(os.path.join(ROOT, "include", "gpmap.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(gp_[a-z0-9_]+)\s*\(", header))
    assert len(declared) >= 20
    for name in declared:
        assert hasattr(L, name), "libgpmap.so does not export %s" % name
    assert declared == set(gpmap.SIGNATURES), declared ^ set(gpmap.SIGNATURES)


def test_library_contains_sm100a_tensor_core_code():
    """The BUILT library holds sm_100a tensor-core machine code: cuobjdump of libgpmap.so must show the int8 tcgen05
    MMA (UTCIMMA), TMEM loads (LDTM), TMA bulk copies (UBLKCP) and tcgen05 commits (UTCBAR) in the scoring kernels."""
    import shutil
    import subprocess
    path = gbuild.build()
    tool = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    sass = subprocess.run([tool, "-sass", path], capture_output=True, text=True, check=True).stdout
    assert "sm_100a" in sass
    counts = {op: len(re.findall(r"\b%s\b" % op, sass)) for op in ("UTCIMMA", "LDTM", "UBLKCP", "UTCBAR")}
    assert all(v > 0 for v in counts.values()), counts
    kernels = re.findall(r"Function : (\S+)", sass)
    assert any("scoring_kernel" in k for k in kernels) and any("sequence_kernel" in k for k in kernels)
    assert any("mma_probe_kernel" in k for k in kernels)


def test_tuning_and_map_units_host_side():
    """gp_tuning round trip and the unit table of gp_enumerate_map_range (host logic, no GPU): units are the m <= rev m,
    pairs first; every genotype of the map belongs to exactly one unit."""
    S = gpmap.Structures(4, 4)
    assert S.tuning() == dict(fold_bits=15, sym_bits=7, narrow_rows=1, seq_tensor=1)
    for bad in (dict(fold_bits=8), dict(fold_bits=23), dict(sym_bits=4), dict(sym_bits=12), dict(narrow_rows=2), dict(seq_tensor=3)):
        with pytest.raises(gpmap.GpError) as ei:
            S.tune(**bad)
        assert ei.value.status == 1 and S.tuning()["fold_bits"] == 15
    for k in (5, 6, 7, 8):
        S.tune(sym_bits=k)
        U = S.map_units()
        mid = 16 - 2 * k
        ms = [S.map_unit(u) for u in range(U)]
        assert all(kk == k for _, kk in ms)
        rev = lambda m: int(format(m, "0%db" % mid)[::-1], 2) if mid else 0
        pal = [m for m, _ in ms if rev(m) == m]
        assert [m for m, _ in ms][len(ms) - len(pal):] == sorted(pal) and len(pal) == 1 << ((mid + 1) // 2)
        assert sorted([m for m, _ in ms] + [rev(m) for m, _ in ms if rev(m) != m]) == list(range(1 << mid))
        g = S.map_range_genotypes(0, U)
        assert g.size == 1 << 16 and np.array_equal(np.sort(g), np.arange(1 << 16, dtype=np.uint64))
        assert int(gpmap.lib().gp_map_range_genotypes(S._h, 0, U)) == 1 << 16
        assert int(gpmap.lib().gp_map_range_genotypes(S._h, U, 1)) == 0
    S.close()
    S3 = gpmap.Structures(3, 3)                 # N = 9: too short for the scheme, one unit = the whole map
    assert S3.map_units() == 1 and S3.map_unit(0) == (0, 0)
    assert int(gpmap.lib().gp_map_range_genotypes(S3._h, 0, 1)) == 512
    S3.close()
    S6 = gpmap.Structures(6, 6)
    assert S6.map_units() == (1 << 21) + (1 << 10)
    S6.close()


def test_status_strings_and_tile():
    L = gpmap.lib()
    assert L.gp_strerror(0) == b"ok"
    assert all(L.gp_strerror(i) for i in range(7)) and b"scratch" in L.gp_strerror(6)
    assert gpmap.tile() == 512


@pytest.mark.parametrize("dims", [(2, 2, 1), (3, 3, 1), (3, 2, 1), (4, 4, 1), (5, 5, 1), (2, 2, 2), (4, 3, 1), (6, 6, 1),
                                  (3, 3, 3)])
def test_structures_match_oracle(oracle_structures, dims):
    S = gpmap.Structures(*dims)
    O = oracle_structures(*dims)
    assert (S.N, S.D, S.C, S.NBP, S.self_reverse, S.walk_count) == (O.N, O.D, O.C, O.NBP, O.self_reverse, O.walk_count)
    step = max(1, S.D // 2000)
    for d in list(range(0, S.D, step)) + [S.D - 1]:
        s1, c1, k1 = S.get(d)
        s2, c2, k2 = O.get(d)
        assert np.array_equal(s1, s2) and np.array_equal(c1, c2) and k1 == k2, (dims, d)
    S.close()


def test_structure_counts_are_the_papers():
    pins = read_pins()
    S = gpmap.Structures(6, 6)
    assert S.D == pins["folds_6x6_directed"] and S.N == pins["length_6x6"]
    assert S.K == 325 and S.NBP == 25
    S.close()


def test_bad_arguments():
    L = gpmap.lib()
    h = ctypes.c_void_p()
    assert L.gp_structures(0, 3, 1, ctypes.byref(h)) == 2 and not h.value
    assert L.gp_structures(9, 9, 1, ctypes.byref(h)) == 2
    assert L.gp_structures(3, 3, 1, None) == 1
    S = gpmap.Structures(3, 3)
    assert L.gp_structures_get(S._h, S.D, None, None, None) == 5
    # compute calls on a handle without device tables report a CUDA error instead of falling back (no GPU here)
    import torch
    if not torch.cuda.is_available():
        en = gpmap._energies(gpmap.HP_ENERGIES, 2, 1)
        dummy = ctypes.c_void_p(16)
        assert L.gp_enumerate(S._h, ctypes.byref(en), 0, 512, dummy, None, None) == 4
        assert L.gp_enumerate_simple(S._h, ctypes.byref(en), 0, 512, dummy, None, None) == 4
    en = gpmap._energies((0, -10, -11, -23), 2, 1)  # asymmetric
    assert L.gp_enumerate(S._h, ctypes.byref(en), 0, 512, ctypes.c_void_p(16), None, None) == 1
    en = gpmap._energies((0, -100, -100, -23), 2, 1)  # weights beyond int8
    assert L.gp_enumerate(S._h, ctypes.byref(en), 0, 512, ctypes.c_void_p(16), None, None) == 1
    en = gpmap._energies((0, -10, -10, -60), 2, 1)    # lin and quad fit, their sum over three contacts does not
    assert L.gp_enumerate(S._h, ctypes.byref(en), 0, 512, ctypes.c_void_p(16), None, None) == 1
    assert L.gp_enumerate_map_range(S._h, ctypes.byref(en), 0, 1, ctypes.c_void_p(16), None, 0, None) == 1
    en = gpmap._energies(gpmap.HP_ENERGIES, 2, 0)  # threshold < 1
    assert L.gp_enumerate(S._h, ctypes.byref(en), 0, 512, ctypes.c_void_p(16), None, None) == 1
    en = gpmap._energies(gpmap.HP_ENERGIES, 2, 1)
    assert L.gp_enumerate(S._h, ctypes.byref(en), 100, 12, ctypes.c_void_p(16), None, None) == 5  # misaligned
    assert L.gp_enumerate(S._h, ctypes.byref(en), 0, 513, ctypes.c_void_p(16), None, None) == 5  # beyond 2^9
    S.close()


def test_seeded_generator_matches_recipe():
    """DESIGN.md section 4 is implemented twice (oracle, library); both must produce the same stream."""
    for seed in (200805612, 1, 2 ** 63 + 5):
        assert np.array_equal(gpmap.seeded_matrix(seed), orc.seeded_matrix(seed))
        assert np.array_equal(gpmap.seeded_sequences(seed, 12345, 300, 16), orc.seeded_sequences(seed, 12345, 300, 16))
        assert np.array_equal(gpmap.seeded_sequences(seed, 1 << 40, 50, 36), orc.seeded_sequences(seed, 1 << 40, 50, 36))
        for alphabet in (2, 3, 20):
            assert np.array_equal(gpmap.seeded_letters(seed, 999, 200, 36, alphabet), orc.seeded_letters(seed, 999, 200, 36, alphabet))
    assert gpmap.lib().gp_seeded_letters(1, 0, 1, 16, 21, np.zeros(16, np.uint8).ctypes.data_as(gpmap._u8p)) == 1
    M = gpmap.seeded_matrix(200805612)
    assert M.min() >= -750 and M.max() <= -50 and np.array_equal(M, M.T)


def test_full_map_resume_fails_loudly_without_a_saved_store(tmp_path):
    """full_map --resume never restarts silently (host logic; the checks come before any device work): no progress file,
    a progress file of a run with other settings, and a run that saved no store are all errors."""
    import json
    from paper_2008_05612_b200 import full_map
    out = str(tmp_path / "map")
    with pytest.raises(RuntimeError, match="does not exist"):
        full_map.run("4x4", out, chunks=4, resume=True)
    S = gpmap.Structures(4, 4)
    U = S.map_units()
    S.close()
    assert U >= 3
    prog = {"lattice": "4x4", "chunks": 2, "units": U, "prefix_path": False, "chunks_done": 1, "store_saved": False}
    with open(os.path.join(out, "progress.json"), "w") as f:
        json.dump(prog, f)
    with pytest.raises(RuntimeError, match="saved no store"):
        full_map.run("4x4", out, chunks=2, resume=True)
    with pytest.raises(RuntimeError, match="other settings"):
        full_map.run("4x4", out, chunks=3, resume=True)
