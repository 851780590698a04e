#!/usr/bin/env python
"""bench.py — throughput of the GP-map hot path on B200.

A step = one pass of the whole hot path over one batch: a genotype-prefix tile of 2^G consecutive 6x6 HP genotypes
(default G = 26; BASELINE.json configs[3] is processed "in genotype-prefix tiles") scored on all 57 337 directed 6x6
structures (a1-a4: tcgen05 int8 contraction + fused argmin-with-uniqueness, uint16 phenotypes into HBM), then the
designability histogram (a5) and the one-point-mutation neighbour pass with the pair bitmap (a6) over the tile's own
G mutable bits.  Every step takes a different seeded prefix, so nothing is cached between steps; the tile's phenotype
store (2^G x 2 B = 134 MB at G = 26) and its weight images (0.9 GB) are larger than the 126 MB L2.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--log2-genotypes G] [--lattice 6x6|5x5|3x3x3|4x4]
  python bench.py --impl reference ...     # the CPU oracle, as it stands, on a bounded sample of the same workload
  python bench.py --full                   # one step = the whole 2^36 map (137 GB store); long
  python bench.py --rows                   # every row of SURVEY.md section 8(a) on its own configuration
The default run also enumerates the WHOLE 6x6 map once (gp_enumerate_map_range in chunks + designability + neighbour
pass over the resident 137 GB store, about 2 minutes; --no-full-map skips it) and prints its measured wall time.

N > 1 (torchrun): each rank takes its own prefix tiles (genotype ranges are independent); no
data-path collective; value = evaluations of all ranks / max-over-ranks device time ("weak" scaling).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "genotype x structure energy evals/s (6x6 HP prefix tile; the full 2^36 enumeration is timed live beside it)"
UNIT = "evals/s"
LATTICES = {"4x4": (4, 4, 1), "5x5": (5, 5, 1), "3x3x3": (3, 3, 3), "6x6": (6, 6, 1)}
SEED = 200805612


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--lattice", default="6x6", choices=sorted(LATTICES))
    ap.add_argument("--log2-genotypes", type=int, default=26, help="genotypes per step = 2^G (clamped to the map)")
    ap.add_argument("--full", action="store_true", help="one step = the full map of the lattice")
    ap.add_argument("--cpu-seconds", type=float, default=10.0, help="target CPU time of the oracle sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-whole-map", action="store_true", help="skip the whole-3x3x3-map leg")
    ap.add_argument("--no-full-map", action="store_true", help="skip the live full 2^36 6x6 enumeration leg (about 2 minutes)")
    ap.add_argument("--fold-bits", type=int, default=0, help="gp_tuning.fold_bits: low genotype bits kept as MMA columns")
    ap.add_argument("--force-sharded", action="store_true", help="take the sharded multi-rank step (sharding.py over "
                    "torch.distributed) even with one rank: exercises that code path on a single GPU")
    ap.add_argument("--map-units", type=int, default=0, help="time gp_enumerate_map_range on this many units of the map (compact "
                                                             "layout, no full store) instead: the map path's kernels on their own")
    ap.add_argument("--rows", action="store_true", help="time every row of the hot path on its BASELINE.json config instead")
    ap.add_argument("--out", default="", help="--rows: also write the rows to this JSON file")
    return ap.parse_args()


def tile_begin(step, rank, world, G, N):
    """First genotype of the prefix tile of (step, rank): seeded, distinct per step and rank."""
    import numpy as np
    n_tiles = 1 << (N - G)
    if n_tiles == 1:
        return 0
    rng = np.random.default_rng(SEED)
    perm_seed = int(rng.integers(1, 1 << 30)) | 1
    idx = ((step * world + rank) * 2654435761 + perm_seed) % n_tiles
    return idx << G


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.thread.join(timeout=2)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except ValueError:
                continue
            for nm, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "power_w_max": max(pw), "samples": len(sm),
                "reasons": sorted(reasons)}


def peaks():
    """(hbm GB/s, bf16 burst TF/s, bf16 sustained TF/s, source) from MEASURED_PEAKS.json, else the guide's fallback."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), float(p["bf16_tflops"]), float(p.get("bf16_tflops_sustained", p["bf16_tflops"])), "measured"
    except (OSError, KeyError, ValueError):
        return 6650.0, 1590.0, 1400.0, "fallback"




PROFILE_CSV = os.path.join(ROOT, "profiles", "r3_scoring_ncu_raw.csv")


ROB_WARP_INSTR_PER_FLIP = 0.285   # profiles/r2_robustness_ncu.md: (2.69e8 + 2.29e8) warp instructions / (2^26 x 26 genotype-flips)


def folded_columns(mon):
    """Contraction columns the scoring kernel executes when the monomers `mon` stay free inside one weight image
    (DESIGN.md 6.1): 2 bias columns + the monomers + the monomer pairs that can touch (odd distance >= 3)."""
    return 2 + len(mon) + sum(1 for i in range(len(mon)) for j in range(i + 1, len(mon))
                              if mon[j] - mon[i] >= 3 and (mon[j] - mon[i]) % 2 == 1)


def image_bytes(columns, k_exec, narrow_rows):
    """Bytes of ONE weight image in HBM: 128-row tiles over the structure columns, rows of 64 bytes when the folded
    contraction fits them (gp_tuning.narrow_rows), else 128 bytes per 128 features."""
    row = 64 if (narrow_rows and k_exec <= 64) else 128 * ((k_exec + 127) // 128)
    return ((columns + 127) // 128) * 128 * row


def ncu_profile():
    """Tensor-pipe activity and DRAM bytes of one scoring_kernel launch from the committed `ncu --page raw --csv` export
    (profiles/r3_scoring_ncu_raw.csv; the command is in profiles/r3_scoring_ncu.md): taken under the profiler in a
    separate run of the same configuration, read here by file parse only.  None if the file is absent."""
    import csv
    try:
        with open(PROFILE_CSV, newline="") as f:
            rows = [r for r in csv.reader(f) if r]
    except OSError:
        return None
    head = next((r for r in rows if "Kernel Name" in r), None)
    if head is None:
        return None
    body = [r for r in rows[rows.index(head) + 1:] if len(r) == len(head)]
    vals = next((r for r in body if "scoring_kernel" in r[head.index("Kernel Name")]), None)
    units = body[0] if body and body[0][head.index("Kernel Name")] == "" else None
    if vals is None:
        return None

    def get(name, scale_by_unit=True):
        if name not in head:
            return None
        i = head.index(name)
        v = float(vals[i].replace(",", ""))
        if scale_by_unit and units:
            v *= {"Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "byte": 1.0, "ms": 1.0, "us": 1e-3, "ns": 1e-6}.get(units[i], 1.0)
        return v
    rd, wr = get("dram__bytes_read.sum"), get("dram__bytes_write.sum")
    return {"file": os.path.relpath(PROFILE_CSV, ROOT), "kernel": vals[head.index("Kernel Name")],
            "tensor_active_pct": get("sm__pipe_tensor_subpipe_imma_cycles_active.avg.pct_of_peak_sustained_active", False),
            "alu_active_pct": get("sm__pipe_alu_cycles_active.avg.pct_of_peak_sustained_active", False),
            "duration_ms": get("gpu__time_duration.sum"),
            "dram_bytes": (rd + wr) if rd is not None and wr is not None else None}


def _oracle_range(args):
    dims, begin, count = args
    from oracle import gp_oracle as orc
    O = _oracle_range.cache.setdefault(dims, None) or orc.Structures(*dims)
    _oracle_range.cache[dims] = O
    t0 = time.perf_counter()
    O.enumerate(begin, count, want_gap=False)
    return time.perf_counter() - t0


_oracle_range.cache = {}


def oracle_rate(dims, begins, seconds, O=None):
    """evals/s of the oracle as it stands, 1 thread: consecutive genotypes from each of `begins`, about `seconds` in all."""
    from oracle import gp_oracle as orc
    O = O or orc.Structures(*dims)
    total = 1 << O.N
    n = min(64, total)
    O.enumerate(begins[0], n, want_gap=False)  # page in
    t0 = time.perf_counter()
    O.enumerate(begins[0], n, want_gap=False)
    per = max(time.perf_counter() - t0, 1e-7) / n
    each = int(max(1, min(total, seconds / per) // len(begins)))
    done, t0 = 0, time.perf_counter()
    for b in begins:
        c = min(each, total - b)
        O.enumerate(b, c, want_gap=False)
        done += c
    dt = time.perf_counter() - t0
    return done * O.D / dt, dt, done, O


def cpu_baseline(dims, begins, cpu_seconds, G, N):
    """the oracle, as it stands, on this box's host cores.  `value` = 1 thread on the bench
    workload (config 4); the other configs, the all-core aggregate (independent processes on disjoint ranges) and the
    oracle's neighbour pass are listed beside it."""
    import numpy as np
    from oracle import gp_oracle as orc
    v, secs, done, O = oracle_rate(dims, begins, cpu_seconds)
    out = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "seconds": secs,
           "sample": "%d ranges x %d consecutive genotypes of the step's tiles x %d structures (%.3g evals), 1 thread"
                     % (len(begins), done // len(begins), O.D, done * O.D),
           "host_cores_available": os.cpu_count(), "full_6x6_map_extrapolated_s": float(1 << 36) * 57337 / v if dims == (6, 6, 1) else None}
    # all cores: one process per core, each its own disjoint range of the same tile (fork: the fold library is shared)
    try:
        import multiprocessing as mp
        cores = os.cpu_count() or 1
        per = max(64, done)                      # every process does as much as the single-thread sample did in all
        _oracle_range.cache[dims] = O
        jobs = [(dims, begins[i % len(begins)] + (1 + i // len(begins)) * per * 4, per) for i in range(cores)]
        with mp.get_context("fork").Pool(cores) as pool:
            t0 = time.perf_counter()
            pool.map(_oracle_range, jobs)
            wall = time.perf_counter() - t0
        out["all_cores"] = {"value": cores * per * O.D / wall, "unit": UNIT, "cores": cores, "seconds": wall,
                            "sample": "%d processes x %d genotypes" % (cores, per)}
    except Exception as e:  # a box that cannot fork is not a bench failure
        out["all_cores"] = {"unavailable": repr(e)}
    others = {}
    for name, d, b, secs_each in (("config1_4x4_full_map", (4, 4, 1), [0], None), ("config2_5x5", (5, 5, 1), [0, 21 << 20], 3.0),
                                  ("config3_3x3x3", (3, 3, 3), [0, 0x2B5 << 16, (1 << 27) - (1 << 12)], 3.0)):
        if secs_each is None:
            Od = orc.Structures(*d)
            t0 = time.perf_counter()
            Od.enumerate(0, 1 << Od.N, want_gap=False)
            dt = time.perf_counter() - t0
            others[name] = {"evals_per_s": float(1 << Od.N) * Od.D / dt, "seconds": dt, "genotypes": 1 << Od.N}
        else:
            r, dt, dn, Od = oracle_rate(d, b, secs_each)
            others[name] = {"evals_per_s": r, "seconds": dt, "genotypes": dn}
    O4 = orc.Structures(4, 4)
    n5 = 1 << 20
    seqs = orc.seeded_sequences(SEED, 0, n5, 16)
    M = orc.seeded_matrix(SEED)
    t0 = time.perf_counter()
    O4.enumerate_seqs(seqs, M, 20, want_gap=False)
    dt = time.perf_counter() - t0
    others["config5_mj4x4"] = {"evals_per_s": n5 * O4.D / dt, "seconds": dt, "sequences": n5}
    # neighbour pass of the oracle over a store shaped like config 2 (549 classes, 63 % null; seeded), a quarter of its
    # size so that the sample stays bounded: 2^23 entries x 23 flips
    rng = np.random.default_rng(SEED)
    store = rng.integers(0, 549, size=1 << 23).astype(np.uint16)
    store[rng.random(1 << 23) < 0.63] = 0xFFFF
    t0 = time.perf_counter()
    orc.robustness(store, 23, 549)
    dt = time.perf_counter() - t0
    others["neighbour_pass_config2_shape"] = {"seconds": dt, "genotypes": 1 << 23, "genotype_flips_per_s": float(23 << 23) / dt,
                                              "store": "seeded synthetic, 549 classes, 63 % null"}
    out["other_configs"] = others
    return out


def run_reference(args):
    """--impl reference: the oracle on the box's host cores, same config/metric; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    dims = LATTICES[args.lattice]
    N = dims[0] * dims[1] * dims[2]
    G = N if args.full else min(args.log2_genotypes, N)
    from oracle import gp_oracle as orc
    O = orc.Structures(*dims)
    # one "step" = a bounded sample of the step's prefix tile: the first `m` genotypes of the tile
    per_step_seconds = max(1.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    t0 = time.perf_counter()
    O.enumerate(0, 64, want_gap=False)
    per = max(time.perf_counter() - t0, 1e-6) / 64
    m = int(max(64, min(1 << G, per_step_seconds / per)))
    times = []
    for step in range(args.warmup + args.steps):
        b = tile_begin(step, 0, 1, G, N)
        t0 = time.perf_counter()
        ph = O.enumerate(b, m, want_gap=False)
        orc.designability(ph, O.C)
        dt = time.perf_counter() - t0
        if step >= args.warmup:
            times.append(dt)
    tot = sum(times)
    value = m * O.D * len(times) / tot
    sample = "first %d genotypes of each step's 2^%d-genotype tile x %d structures, 1 thread" % (m, G, O.D)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot / len(times), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int32", "data": "synthetic",
            "config": workload_config(args.lattice, G, O.D, O.C, O.N + sum(1 for i in range(O.N) for j in range(i + 3, O.N, 2)), 1 << G,
                                      full=args.full),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def workload_config(lattice, G, D, C, K, n, parallelism="independent prefix tiles per rank, no collective", full=False):
    """The `config` object: identical keys in both arms."""
    return {"workload": ("%s HP whole map (reversal identity): 2^%d genotypes x %d directed structures, then designability + "
                         "neighbour pass" if full else
                         "%s HP genotype-prefix tile: 2^%d genotypes x %d directed structures, then designability + "
                         "neighbour pass over the tile") % (lattice, G, D),
            "lattice": lattice, "log2_genotypes": G, "D": D, "C": C, "features_K": K,
            "l2": "inputs larger than L2 (per step: %.0f MB phenotype tile, fresh seeded prefix, weight images rebuilt)"
                  % (2.0 * n / 1e6),
            "parallelism": parallelism}


def full_map_leg(lattice, stream, cpu_check=True):
    """BASELINE.json configs[3] live: the WHOLE map of the lattice through gp_enumerate_map_range (chunks of units, so the
    run can report progress and could resume), gp_reduce_store over the resident store; device
    times from CUDA events on the launching stream; invariants; a seeded sample of phenotypes against the oracle."""
    import numpy as np
    import torch
    from paper_2008_05612_b200 import gpmap
    S = gpmap.Structures(*LATTICES[lattice])
    N, D, C = S.N, S.D, S.C
    total = 1 << N
    free, _ = torch.cuda.mem_get_info()
    need = 2 * total + (3 << 30)
    if free < need:
        return {"skipped": "needs %.1f GB of free HBM, %.1f GB free" % (need / 1e9, free / 1e9)}
    pheno = torch.empty(total, dtype=torch.uint16, device="cuda")
    U = S.map_units()
    chunks = 64 if U >= 64 else 1
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    l0 = gpmap.launch_count()
    gpmap.kernel_timing(True)
    for w in range(4):
        gpmap.kernel_time(w)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    ev[0].record(stream)
    for c in range(chunks):
        u0, u1 = U * c // chunks, U * (c + 1) // chunks
        S.enumerate_map_range(u0, u1 - u0, pheno, stream=stream)
    ev[1].record(stream)
    hist, R, Dl, Oc, pairs = gpmap.reduce_store(pheno, N, C, stream=stream)   # a5 + a6: designability from the first sweep
    ev[2].record(stream)
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    t_score, t_red = (ev[i].elapsed_time(ev[i + 1]) * 1e-3 for i in range(2))
    launches = gpmap.launch_count() - l0
    ktime = [gpmap.kernel_time(w) for w in range(4)]
    gpmap.kernel_timing(False)
    hist = hist.cpu().numpy().astype(np.uint64)
    R, Dl, Oc = (x.cpu().numpy().astype(np.uint64) for x in (R, Dl, Oc))
    folding = int(hist[:C].sum())
    # the tiled neighbour pass on this store runs geometries the oracle cannot reach (third pass): gp_phi_row, an
    # untiled kernel of its own, is the independent witness (row[q] = R[q], sum_{p != q} row[p] = O[q], row[C] = D[q])
    from paper_2008_05612_b200.full_map import phi_row_witness
    witness = phi_row_witness(gpmap, pheno, N, C, hist, R, Dl, Oc)
    # map-path roofline of the scoring phase as a whole (image builds, combines and launch tails included): executed int8
    # ops of the folded contraction over the device time of the phase, against the MMA-only probe of the same K steps
    k = min(S.tuning()["sym_bits"], N // 2)
    k_exec = folded_columns(list(range(k)) + list(range(N - k, N)))
    k_steps = (k_exec + 31) // 32
    probe_ops, probe_clk, probe_mhz = gpmap.probe_i8_peak(k_steps, 1.0)
    achieved = 2.0 * k_exec * float(total) * C / t_score / 1e12
    sc_ms, sc_n = ktime[gpmap.KERNEL_SCORING]
    im_ms, im_n = ktime[gpmap.KERNEL_IMAGE]
    img_b = image_bytes(C, k_exec, S.tuning()["narrow_rows"])
    n_images = float(total) / float(1 << (2 * k))
    map_roofline = {"kernel": "tc::scoring_kernel (hrec mode) + tc::build_image_kernel + tc::combine_kernel, whole scoring phase",
                    "bound": "tensor", "achieved": achieved, "peak": probe_ops / 1e12, "unit": "TFLOP/s",
                    "frac": achieved / (probe_ops / 1e12), "traffic": None,
                    "peak_source": "gp_probe_i8_peak(k_steps=%d), measured after the map" % k_steps,
                    "ops_per_eval_executed": 2.0 * k_exec, "ops_per_eval_issued": 64.0 * k_steps,
                    "frac_issued": achieved * 32.0 * k_steps / k_exec / (probe_ops / 1e12),
                    "algorithmic_bytes": 2.0 * total, "image_bytes": 2.0 * n_images * img_b,
                    "scoring_launches": int(sc_n), "scoring_launch_ms_summed": sc_ms, "image_launches": int(im_n),
                    "image_launch_ms_summed": im_ms,
                    "note": "launches of a range alternate between two streams and overlap, so the summed per-launch times "
                            "may exceed the phase time; the fraction uses the phase time"}
    rng = np.random.default_rng(SEED)
    g = rng.integers(0, total, size=1 << 20, dtype=np.uint64)
    rev = np.zeros_like(g)
    for i in range(N):
        rev |= ((g >> np.uint64(i)) & np.uint64(1)) << np.uint64(N - 1 - i)
    s16 = pheno.view(torch.int16)
    rev_bad = int((s16[torch.from_numpy(g.astype(np.int64)).cuda()] != s16[torch.from_numpy(rev.astype(np.int64)).cuda()]).sum())
    out = {"workload": "%s HP whole map: 2^%d genotypes x %d directed structures (%d representatives scored, reversal "
                       "identity), uint16 store resident in HBM (%.1f GB), designability + neighbour pass + pair count"
                       % (lattice, N, D, C, 2.0 * total / 1e9),
           "wall_s": wall, "device_s": {"scoring": t_score, "designability_and_neighbour_pass": t_red, "total": t_score + t_red},
           "effective_evals_per_s": float(total) * D / t_score, "executed_evals_per_s": float(total) * C / t_score,
           "store_GBps": {"reduce_store_algorithmic": 2.0 * total / t_red / 1e9},
           "roofline": map_roofline,
           "gpu_launches": int(launches), "unit_chunks": chunks,
           "folding": folding, "folding_fraction": folding / total, "designable_classes": int((hist[:C] > 0).sum()),
           "phenotype_pairs": int(pairs.item()), "sum_R": int(R.sum()), "sum_D": int(Dl.sum()), "sum_O": int(Oc.sum()),
           "invariants": {"hist_sums_to_2^N": int(hist.sum()) == total,
                          "R+D+O_equals_N_x_folding": int(R.sum() + Dl.sum() + Oc.sum()) == N * folding,
                          "sum_R_even": int(R.sum()) % 2 == 0, "sum_O_even": int(Oc.sum()) % 2 == 0,
                          "reversal_symmetry_mismatches_of_2^20": rev_bad}}
    out["invariants"].update(witness)
    if cpu_check:
        from oracle import gp_oracle as orc
        O = orc.Structures(*LATTICES[lattice])
        bad = n_chk = 0
        for b in [0, total - 256] + [int(x) for x in rng.integers(0, total - 256, size=6)]:
            want = O.enumerate(b, 256, want_gap=False)
            bad += int((pheno[b:b + 256].cpu().numpy() != want).sum())
            n_chk += 256
        out["oracle_sampled"] = {"genotypes": n_chk, "mismatches": bad}
    del pheno
    S.close()
    torch.cuda.empty_cache()
    return out


def run_map_units(args):
    """--map-units U: `steps` calls of gp_enumerate_map_range over U units of the lattice's map in the compact layout
    (a slice of the whole-map run that needs no 2^N store), after `warmup` calls; CUDA-event time.  The committed command
    behind the map-path ncu captures under profiles/."""
    import torch
    from paper_2008_05612_b200 import gpmap
    S = gpmap.Structures(*LATTICES[args.lattice])
    U = min(args.map_units, S.map_units())
    first = (S.map_units() - U) // 3
    n = int(gpmap.lib().gp_map_range_genotypes(S._h, first, U))
    ph = torch.empty(n, dtype=torch.uint16, device="cuda")
    for _ in range(args.warmup):
        S.enumerate_map_range(first, U, ph, compact=True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(args.steps):
        S.enumerate_map_range(first, U, ph, compact=True)
    e1.record()
    torch.cuda.synchronize()
    t = e0.elapsed_time(e1) * 1e-3 / args.steps
    print(json.dumps({"row": "f1 gp_enumerate_map_range (compact layout)", "lattice": args.lattice, "units": U, "first_unit": first,
                      "genotypes": n, "seconds_per_call": t, "executed_evals_per_s": float(n) * S.C / t,
                      "effective_evals_per_s": float(n) * S.D / t, "sym_bits": S.tuning()["sym_bits"]}), flush=True)
    S.close()


def run_rows(args):
    """--rows: every row of SURVEY.md section 8(a) on the configuration BASELINE.json names for it (CUDA-event times
    after one warm-up call; a0 is host wall time).  Prints one JSON object per row."""
    import numpy as np
    import torch
    from paper_2008_05612_b200 import gpmap

    def dev_time(fn, reps=2):
        fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) * 1e-3 / reps

    rows, structs = [], {}
    for name in ("4x4", "5x5", "3x3x3", "6x6"):
        t0 = time.perf_counter()
        structs[name] = gpmap.Structures(*LATTICES[name])
        rows.append(dict(row="a0 gp_structures", config=name, seconds=time.perf_counter() - t0,
                         note="D=%d C=%d" % (structs[name].D, structs[name].C)))
    for name in ("4x4", "5x5", "3x3x3"):
        S = structs[name]
        n = 1 << S.N
        ph = torch.empty(n, dtype=torch.uint16, device="cuda")
        gap = torch.empty(n, dtype=torch.int16, device="cuda")
        t = dev_time(lambda: S.enumerate(0, n, ph))
        rows.append(dict(row="a1-a4 gp_enumerate (prefix path, D columns)", config=name, seconds=t, evals_per_s=n * S.D / t))
        t = dev_time(lambda: S.enumerate_map(ph, gap))
        rows.append(dict(row="a1-a4 gp_enumerate_map (reversal identity, C columns)", config=name, seconds=t,
                         effective_evals_per_s=n * S.D / t))
        m = min(n, 1 << 22)
        t = dev_time(lambda: S.enumerate(0, m, ph, simple=True), reps=1)
        rows.append(dict(row="a1-a4 gp_enumerate_simple (CUDA cores)", config=name + " first 2^22", seconds=t, evals_per_s=m * S.D / t))
        S.enumerate_map(ph, gap)
        t = dev_time(lambda: gpmap.designability(ph, S.C))
        rows.append(dict(row="a5 gp_designability", config=name, seconds=t, GBps=2.0 * n / t / 1e9))
        t = dev_time(lambda: gpmap.robustness(ph, S.N, S.C))
        rows.append(dict(row="a6 gp_robustness (+ pair bitmap)", config=name, seconds=t, GBps_algorithmic=2.0 * n / t / 1e9))
        t = dev_time(lambda: gpmap.nn_components(ph, S.N, S.C), reps=1)
        rows.append(dict(row="a7 gp_nn_components", config=name, seconds=t))
        t = dev_time(lambda: gpmap.threshold_sweep(ph, gap, S.C, [1, 2, 3, 10, 24]))
        rows.append(dict(row="f4 gp_threshold_sweep (5 thresholds)", config=name, seconds=t, GBps=4.0 * n / t / 1e9))
        del ph, gap
    for name, paper_hp, paper_mj in (("6x6", 1.35e-4, 1.19e-4), ("3x3x3", 2.6e-4, 2.8e-4)):  # PAPER.md:195-204 Table 3
        S = structs[name]
        cnt = 1 << 21
        seqs = torch.from_numpy(np.random.default_rng(SEED).integers(0, 2, size=(cnt, S.N), dtype=np.uint8)).cuda()
        ph = torch.empty(cnt, dtype=torch.uint16, device="cuda")
        e = np.array(gpmap.HP_ENERGIES, np.int32)
        for label, on, c in (("tensor cores", 1, cnt), ("CUDA cores", 0, 1 << 17)):
            S.tune(seq_tensor=on)
            t = dev_time(lambda: S.enumerate_seqs(seqs[:c], ph[:c], None, e=e, alphabet=2), reps=1)
            rows.append(dict(row="f3 sampling, random HP sequences (%s)" % label, config="%s, %d sequences" % (name, c), seconds=t,
                             evals_per_s=c * S.D / t, seconds_per_sequence=t / c, paper_gpu_seconds_per_sequence=paper_hp))
        S.tune(seq_tensor=1)
        t = dev_time(lambda: S.enumerate_seeded(SEED, 0, cnt, ph, e=e, alphabet=2), reps=1)
        rows.append(dict(row="f3 sampling, seeded HP sequences drawn on chip (tensor cores)", config="%s, %d sequences" % (name, cnt),
                         seconds=t, evals_per_s=cnt * S.D / t, seconds_per_sequence=t / cnt, paper_gpu_seconds_per_sequence=paper_hp))
        M = gpmap.seeded_matrix(SEED)
        for label, on, c in (("tensor cores, two int8 limbs", 2, 1 << 20), ("CUDA cores", 0, 1 << 17)):
            S.tune(seq_tensor=on)
            t = dev_time(lambda: S.enumerate_seeded(SEED, 0, c, ph[:c], e=M), reps=1)
            rows.append(dict(row="f3 sampling, seeded 20-letter sequences (%s)" % label, config="%s, %d sequences" % (name, c),
                             seconds=t, evals_per_s=c * S.D / t, seconds_per_sequence=t / c,
                             paper_gpu_seconds_per_sequence=paper_mj))
        S.tune(seq_tensor=1)
        del seqs, ph
    S = structs["4x4"]
    M = gpmap.seeded_matrix(SEED)
    n = 1 << 30
    ph = torch.empty(n, dtype=torch.uint16, device="cuda")
    t = dev_time(lambda: S.enumerate_seeded(SEED, 0, n, ph, e=M), reps=1)
    hist = gpmap.designability(ph, S.C)
    rows.append(dict(row="a8 gp_enumerate_seeded (20 letters, seeded matrix; default = CUDA cores at D = 69)", config="4x4, 2^30 sequences",
                     seconds=t, evals_per_s=n * S.D / t, folding_fraction=1.0 - hist[S.C].item() / n))
    S.tune(seq_tensor=2)
    m = 1 << 28
    t = dev_time(lambda: S.enumerate_seeded(SEED, 0, m, ph[:m], e=M), reps=1)
    rows.append(dict(row="a8 gp_enumerate_seeded (20 letters, seeded matrix; forced onto the tensor cores)", config="4x4, 2^28 sequences",
                     seconds=t, evals_per_s=m * S.D / t))
    S.tune(seq_tensor=1)
    for r in rows:
        print(json.dumps(r), flush=True)
    if args.out:
        with open(args.out, "w") as f:
            json.dump(rows, f, indent=1)


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2008_05612_b200 import gpmap

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1 or args.force_sharded:
        if "MASTER_ADDR" not in os.environ:
            os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT="29531", RANK="0", WORLD_SIZE="1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    gpmap.lib()  # fails loudly if libgpmap.so is missing / unbuildable
    if args.rows or args.map_units:
        if rank == 0:
            run_map_units(args) if args.map_units else run_rows(args)
        return

    dims = LATTICES[args.lattice]
    S = gpmap.Structures(*dims)
    if args.fold_bits:
        S.tune(fold_bits=args.fold_bits)
    N, D, C = S.N, S.D, S.C
    G = N if args.full else min(args.log2_genotypes, N)
    n = 1 << G
    pheno = torch.empty(n, dtype=torch.uint16, device="cuda")
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # N > 1: the step is ONE sub-cube of 2^(G+q) genotypes sharded over the ranks on its top q bits:
    # rank-local scoring, rank-local neighbour pass, hypercube exchange of the shards for the q rank-selecting bits,
    # all_reduce of the counts, OR-reduce of the pair bitmap.  Per-rank work is fixed: weak scaling.
    sharded = (world > 1 or args.force_sharded) and (world & (world - 1)) == 0 and G + world.bit_length() - 1 <= N and not args.full
    if sharded:
        from paper_2008_05612_b200 import sharding
        ops, comm, q = sharding.LibOps(), sharding.DistComm(), world.bit_length() - 1

    def step(i):
        if sharded:
            base = tile_begin(i, 0, 1, G + q, N)
            S.enumerate(base + rank * n, n, pheno, stream=stream)                      # a1-a4 on the rank's shard
            return sharding.reduce_store_sharded(ops, comm, pheno, G + q, C)           # a5 + a6 across the shards
        b = tile_begin(i, rank, world, G, N)
        if args.full:
            S.enumerate_map(pheno, stream=stream)                     # a1-a4, whole map through the reversal identity
        else:
            S.enumerate(b, n, pheno, stream=stream)                   # a1-a4
        out = gpmap.reduce_store(pheno, G, C, stream=stream)          # a5 + a6 (+ pair bitmap) in one sweep of the store
        step.hist = out[0]
        return out

    for i in range(args.warmup):
        step(i)
    barrier()
    gpmap.kernel_timing(True)
    for w in range(4):
        gpmap.kernel_time(w)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    l0 = gpmap.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record(stream)
    for i in range(args.steps):
        step(args.warmup + i)
    ev1.record(stream)
    barrier()
    ms = ev0.elapsed_time(ev1)
    clocks = sampler.stop() if rank == 0 else None
    launches = gpmap.launch_count() - l0
    ktime = [gpmap.kernel_time(w) for w in range(4)]
    gpmap.kernel_timing(False)
    if world > 1:
        t = torch.tensor([ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    folding = int(n - step.hist[C].item()) if not sharded else None
    evals_step = float(n) * D * world
    value = evals_step * args.steps / (ms * 1e-3)

    # ---- e2e: the C-ABI call with HOST buffers (pinned output), D2H inside the timed region ----
    e2e = None
    host = torch.empty(n, dtype=torch.uint16).pin_memory() if n <= (1 << 32) else None
    if host is not None:
        host_np = host.numpy()
        e_steps = max(1, args.steps)
        S.enumerate_host(tile_begin(0, rank, world, G, N), n, want_robustness=True, pheno_out=host_np)
        barrier()
        t0 = time.perf_counter()
        for i in range(e_steps):
            S.enumerate_host(tile_begin(args.warmup + i, rank, world, G, N), n, want_robustness=True, pheno_out=host_np)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        if world > 1:
            t = torch.tensor([dt], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        e2e = {"value": evals_step * e_steps / dt, "unit": UNIT, "h2d_bytes_per_step": 16,
               "d2h_bytes_per_step": int(2 * n + 8 * (C + 1) + 24 * C + 8), "steps": e_steps,
               "call": "gp_enumerate_host (host buffers, pinned phenotype output; device store kept in the handle)"}
        del host, host_np

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    hbm, bf16_burst, bf16_sus, src = peaks()
    sc_ms, sc_n = ktime[gpmap.KERNEL_SCORING]
    evals_launch = float(n) * D / max(1, sc_n // max(1, args.steps))  # one rank's launches
    if args.full:                                                     # map path: k free monomers at each chain end, C columns
        k = min(S.tuning()["sym_bits"], N // 2)
        mon = list(range(k)) + list(range(N - k, N))
        evals_launch = float(n) * C / max(1, sc_n // max(1, args.steps))
    else:
        mon = list(range(min(N, S.tuning()["fold_bits"])))            # low genotype bits kept as contraction columns
    k_exec = folded_columns(mon)                                      # bias x2 + monomers + pairs
    k_steps = (k_exec + 31) // 32
    ops_exec = 2.0 * k_exec                                           # int8 multiply-adds x2 of the folded contraction per evaluation
    ops_issued = 2.0 * 32 * k_steps                                   # what the MMAs issue (columns padded to 32-byte K steps)
    dur = sc_ms / max(1, sc_n) * 1e-3
    achieved = ops_exec * evals_launch / dur / 1e12 if dur > 0 else 0.0
    # the peak: this kernel's own MMA stream alone (gp_probe_i8_peak), measured now on this device
    probe_ops, probe_clk, probe_mhz = gpmap.probe_i8_peak(k_steps, 1.0)
    peak_i8 = probe_ops / 1e12
    prof = ncu_profile()
    # the ncu capture describes this run's launches only if it is a launch of the same shape: its duration (cold, under
    # the profiler) must sit near the launch time measured here; otherwise the DRAM figure is dropped, not quoted
    same_shape = bool(prof and prof["duration_ms"] and dur > 0 and 0.8 < prof["duration_ms"] / (dur * 1e3) < 1.35)
    genotypes_launch = evals_launch / (C if args.full else D)
    images_launch = genotypes_launch / float(1 << len(mon))
    img_b = image_bytes(C if args.full else D, k_exec, S.tuning()["narrow_rows"])
    roofline = {"kernel": "tc::scoring_kernel", "bound": "tensor", "achieved": achieved, "peak": peak_i8, "unit": "TFLOP/s",
                "frac": achieved / peak_i8,
                "traffic": prof["dram_bytes"] if same_shape else None,
                "traffic_source": ((prof["file"] + " (one launch under ncu --set full: %.2f ms there, %.2f ms here)"
                                    % (prof["duration_ms"], dur * 1e3)) if same_shape else
                                   ("dropped: the committed capture is not a launch of this shape" if prof else None)),
                # what the DRAM traffic is made of, computed (not profiled): the phenotypes written, and the per-prefix
                # weight images that build_image_kernel writes and this kernel reads back once
                "algorithmic_bytes": 2.0 * genotypes_launch,
                "image_bytes": 2.0 * images_launch * img_b,
                "images_per_launch": images_launch, "bytes_per_image": img_b,
                "peak_source": "gp_probe_i8_peak(k_steps=%d): MMA-only tcgen05.mma kind::i8 stream, measured in this run" % k_steps,
                "peak_i8_measured": {"TOPs": peak_i8, "clk_per_mma": probe_clk, "sm_mhz": probe_mhz},
                "frac_issued": achieved * ops_issued / ops_exec / peak_i8,
                # the MMA-only probe draws more power and runs at a lower SM clock than the scoring kernel does; per clock
                # (probe peak scaled to the clock sampled during the timed region) the issued fraction is what the ncu
                # tensor-pipe-active counter measures
                "frac_issued_per_clock": (achieved * ops_issued / ops_exec / (peak_i8 * clocks["sm_mhz"] / probe_mhz)
                                          if clocks and clocks.get("sm_mhz") and probe_mhz else None),
                "ncu_tensor_active": prof["tensor_active_pct"] / 100.0 if prof and prof["tensor_active_pct"] is not None else None,
                "frac_of_nominal_4500": achieved / 4500.0, "frac_of_2x_bf16_burst": achieved / (2.0 * bf16_burst),
                "frac_of_2x_bf16_sustained": achieved / (2.0 * bf16_sus), "bf16_peaks_source": src,
                "ops_per_eval_executed": ops_exec, "ops_per_eval_issued": ops_issued,
                "ops_per_eval_contraction_as_posed": 2.0 * S.K,
                "avg_launch_ms": dur * 1e3, "launches": int(sc_n),
                "evals_per_s_kernel": evals_launch / dur if dur > 0 else 0.0,
                "share_of_step": sc_ms / ms if ms > 0 else None}
    rb_ms, rb_n = ktime[gpmap.KERNEL_ROBUSTNESS]
    hs_ms, hs_n = ktime[gpmap.KERNEL_HIST]
    im_ms, im_n = ktime[gpmap.KERNEL_IMAGE]
    other = {
        "robustness_kernel": {"bound": "hbm", "algorithmic_GBps": 2.0 * n / (rb_ms / max(1, rb_n) * 1e-3) / 1e9 if rb_ms else None,
                              "peak": hbm, "avg_launch_ms": rb_ms / max(1, rb_n), "share_of_step": rb_ms / ms},
        "hist_kernel": {"bound": "hbm", "algorithmic_GBps": 2.0 * n / (hs_ms / max(1, hs_n) * 1e-3) / 1e9 if hs_ms else None,
                        "peak": hbm, "avg_launch_ms": hs_ms / max(1, hs_n), "share_of_step": hs_ms / ms, "launches": int(hs_n),
                        "note": "the step takes designability from gp_reduce_store (first sweep of the neighbour pass): "
                                "hist_kernel runs only where gp_designability is called on its own"},
        "build_image_kernel": {"avg_launch_ms": im_ms / max(1, im_n), "launches": int(im_n), "share_of_step": im_ms / ms,
                               "note": "runs on a side stream overlapped with the scoring kernel: elapsed, not exclusive, time"},
    }
    for kname in ("robustness_kernel", "hist_kernel"):
        if other[kname]["algorithmic_GBps"]:
            other[kname]["frac_of_hbm"] = other[kname]["algorithmic_GBps"] / hbm
    if rb_ms:
        # the neighbour pass is bound by instruction issue, not HBM.  Peak = 4 schedulers x 148 SMs x one
        # warp instruction per clock at the clock sampled in this run; the kernel's cost is 0.285 warp instructions per
        # genotype-flip (profiles/r2_robustness_ncu.md: 4.98e8 warp instructions for the 2^26 x 26 flips of this tile)
        sm_clk = (clocks or {}).get("sm_mhz") or 1965.0
        issue_peak = 4.0 * 148 * sm_clk * 1e6
        flips_per_s = float(n) * G * args.steps / (rb_ms * 1e-3)
        other["robustness_kernel"].update({"bound": "alu", "unit": "warp instructions/s", "peak": issue_peak,
                                           "achieved": flips_per_s * ROB_WARP_INSTR_PER_FLIP, "frac": flips_per_s * ROB_WARP_INSTR_PER_FLIP / issue_peak,
                                           "genotype_flips_per_s": flips_per_s, "warp_instr_per_flip": ROB_WARP_INSTR_PER_FLIP,
                                           "hbm_peak": hbm})

    whole = None
    if world == 1 and not args.full and not args.no_whole_map:
        # BASELINE.json configs[2]: the paper's fully analysed map, whole, through gp_enumerate_map (reversal identity)
        S3 = gpmap.Structures(3, 3, 3)
        p3 = torch.empty(1 << 27, dtype=torch.uint16, device="cuda")
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps = 3
        for i in range(1 + reps):
            if i == 1:
                torch.cuda.synchronize()
                e0.record(stream)
            S3.enumerate_map(p3, stream=stream)
            h3 = gpmap.reduce_store(p3, 27, S3.C, stream=stream)[0]
        e1.record(stream)
        torch.cuda.synchronize()
        sec = e0.elapsed_time(e1) * 1e-3 / reps
        whole = {"workload": "3x3x3 HP whole map: 2^27 genotypes, 103346 directed structures (51704 scored by the reversal "
                             "identity), designability + neighbour pass", "seconds_per_map": sec,
                 "effective_evals_per_s": float(1 << 27) * S3.D / sec, "executed_evals_per_s": float(1 << 27) * S3.C / sec,
                 "folding": int((1 << 27) - h3[S3.C].item()), "paper_folding_percent": 4.76}
        del p3
        S3.close()

    cpu = None
    if not args.no_cpu_baseline and world == 1:
        begins = [tile_begin(args.warmup + i, 0, 1, G, N) for i in range(min(4, args.steps))]
        cpu = cpu_baseline(dims, begins, args.cpu_seconds, G, N)

    full = None
    if world == 1 and not args.full and not args.no_full_map and args.lattice == "6x6":
        del pheno
        S.close()
        torch.cuda.empty_cache()
        full = full_map_leg("6x6", stream, cpu_check=not args.no_cpu_baseline)

    total_evals_map = float(1 << N) * D
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "s8 x s8 -> s32", "data": "synthetic",
            "config": workload_config(args.lattice, G, D, C, S.K, n, *(["one sub-cube of 2^%d genotypes per step sharded over %d ranks on its top %d "
                                                                        "bits: local scoring, hypercube shard exchange for the neighbour pass "
                                                                        "(%d bytes sent per rank and step), all_reduce of counts, OR-reduce of the "
                                                                        "pair bitmap" % (G + q, world, q, sharding.exchange_bytes_per_rank(G + q, world, C))]
                                                                       if sharded else []), full=args.full),
            "full_map_wall_s_extrapolated_from_tiles": total_evals_map / value * world if value else None,
            "folding_fraction_last_tile": folding / float(n) if folding is not None else None,
            "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline, "other_kernels": other,
            "whole_map_3x3x3": whole, "full_6x6": full, "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)
    if dist.is_initialized():
        dist.destroy_process_group()


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
