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

METRIC = "genotype x structure energy evals/s (6x6 HP prefix tile; full-enumeration wall time extrapolated)"
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
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target CPU time of the oracle sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-whole-map", action="store_true", help="skip the whole-3x3x3-map leg")
    ap.add_argument("--fold-bits", type=int, default=0, help="tuning hook: low genotype bits kept as MMA columns")
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


def oracle_sample(dims, begins, count_each, cpu_seconds):
    """Time the CPU oracle (single thread, as it stands) on genotype ranges of the same workload.
    Returns (evals/s, seconds, description).  The sample grows until it costs about cpu_seconds."""
    from oracle import gp_oracle as orc
    O = orc.Structures(*dims)
    total = 1 << O.N
    n = min(64, total)
    O.enumerate(begins[0], n, want_gap=False)  # page in
    t0 = time.perf_counter()
    O.enumerate(begins[0], n, want_gap=False)
    dt = max(time.perf_counter() - t0, 1e-6)
    per = dt / n
    want = int(max(n, min(total, cpu_seconds / per)))
    per_range = max(1, min(count_each, want // max(1, len(begins))))
    done, t0 = 0, time.perf_counter()
    for b in begins:
        c = min(per_range, total - b)
        O.enumerate(b, c, want_gap=False)
        done += c
    dt = time.perf_counter() - t0
    return done * O.D / dt, dt, "%d ranges x %d consecutive genotypes x %d structures (%.3g evals), 1 thread" % (
        len(begins), per_range, O.D, done * O.D)


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
            "config": {"workload": "%s HP prefix tile, 2^%d genotypes x %d directed structures (oracle sample)" % (
                args.lattice, G, O.D), "lattice": args.lattice, "log2_genotypes": G},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


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
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    gpmap.lib()  # fails loudly if libgpmap.so is missing / unbuildable
    if args.fold_bits:
        gpmap.set_fold_bits(args.fold_bits)

    dims = LATTICES[args.lattice]
    S = gpmap.Structures(*dims)
    N, D, C = S.N, S.D, S.C
    G = N if args.full else min(args.log2_genotypes, N)
    n = 1 << G
    pheno = torch.empty(n, dtype=torch.uint16, device="cuda")
    hist = torch.empty(C + 1, dtype=torch.int64, device="cuda")
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step(i):
        b = tile_begin(i, rank, world, G, N)
        if args.full:
            S.enumerate_map(pheno, stream=stream)                     # a1-a4, whole map through the reversal identity
        else:
            S.enumerate(b, n, pheno, stream=stream)                   # a1-a4
        gpmap.designability(pheno, C, hist=hist, stream=stream)       # a5
        return gpmap.robustness(pheno, G, C, stream=stream)           # a6 (+ pair bitmap)

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
        out = step(args.warmup + i)
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
    folding = int(n - hist[C].item())
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
            r = S.enumerate_host(tile_begin(args.warmup + i, rank, world, G, N), n, want_robustness=True, pheno_out=host_np)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        if world > 1:
            t = torch.tensor([dt], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        e2e = {"value": evals_step * e_steps / dt, "unit": UNIT, "h2d_bytes_per_step": 16,
               "d2h_bytes_per_step": int(2 * n + 8 * (C + 1) + 24 * C + 8), "steps": e_steps,
               "call": "gp_enumerate_host (host buffers, pinned phenotype output; device store kept in the handle)"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    hbm, bf16_burst, bf16_sus, src = peaks()
    sc_ms, sc_n = ktime[gpmap.KERNEL_SCORING]
    evals_launch = float(n) * D / max(1, sc_n // max(1, args.steps))  # one rank's launches
    fb = min(N, args.fold_bits or 15)                                 # low genotype bits kept as contraction columns
    k_exec = 2 + fb + sum(1 for i in range(fb) for j in range(i + 3, fb, 2))  # bias x2 + monomers + pairs
    ops_exec = 2.0 * k_exec                                           # int8 multiply-adds x2 the kernel executes per evaluation
    peak_i8 = 2.0 * bf16_sus                                          # int8 dense = 2 x bf16 (guide's nominal ratio)
    dur = sc_ms / max(1, sc_n) * 1e-3
    achieved = ops_exec * evals_launch / dur / 1e12 if dur > 0 else 0.0
    roofline = {"kernel": "tc::scoring_kernel", "bound": "tensor", "achieved": achieved, "peak": peak_i8, "unit": "TFLOP/s",
                "frac": achieved / peak_i8, "traffic": 965.68e6 * evals_launch / 4.8098e11,
                "traffic_source": "ncu dram__bytes_read+write of profiles/r1_scoring_final_ncu.md, scaled by evaluations per launch",
                "peak_source": "2 x bf16_tflops_sustained (%s); int8 ops" % src,
                "frac_of_nominal_4500": achieved / 4500.0, "frac_of_2x_bf16_burst": achieved / (2.0 * bf16_burst),
                "ops_per_eval_executed": ops_exec, "ops_per_eval_contraction_as_posed": 2.0 * S.K,
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
                        "peak": hbm, "avg_launch_ms": hs_ms / max(1, hs_n), "share_of_step": hs_ms / ms},
        "build_image_kernel": {"avg_launch_ms": im_ms / max(1, im_n), "launches": int(im_n), "share_of_step": im_ms / ms},
    }
    if other["robustness_kernel"]["algorithmic_GBps"]:
        other["robustness_kernel"]["frac"] = other["robustness_kernel"]["algorithmic_GBps"] / hbm
    if other["hist_kernel"]["algorithmic_GBps"]:
        other["hist_kernel"]["frac"] = other["hist_kernel"]["algorithmic_GBps"] / hbm

    cpu = None
    if not args.no_cpu_baseline and world == 1:
        begins = [tile_begin(args.warmup + i, 0, 1, G, N) for i in range(min(4, args.steps))]
        v, secs, desc = oracle_sample(dims, begins, 1 << 20, args.cpu_seconds)
        cpu = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc, "seconds": secs,
               "host_cores_available": os.cpu_count()}

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
            h3 = gpmap.designability(p3, S3.C, stream=stream)
            r3 = gpmap.robustness(p3, 27, S3.C, stream=stream)
        e1.record(stream)
        torch.cuda.synchronize()
        sec = e0.elapsed_time(e1) * 1e-3 / reps
        whole = {"workload": "3x3x3 HP whole map: 2^27 genotypes, 103346 directed structures (51704 scored by the reversal "
                             "identity), designability + neighbour pass", "seconds_per_map": sec,
                 "effective_evals_per_s": float(1 << 27) * S3.D / sec, "executed_evals_per_s": float(1 << 27) * S3.C / sec,
                 "folding": int((1 << 27) - h3[S3.C].item()), "paper_folding_percent": 4.76}
        del p3
        S3.close()
    total_evals_map = float(1 << N) * D
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "s8 x s8 -> s32", "data": "synthetic",
            "config": {"workload": "%s HP genotype-prefix tile: 2^%d genotypes x %d directed structures, then designability + "
                                   "neighbour pass over the tile" % (args.lattice, G, D),
                       "lattice": args.lattice, "log2_genotypes": G, "D": D, "C": C, "features_K": S.K,
                       "l2": "inputs larger than L2 (per step: %.0f MB phenotype tile, fresh seeded prefix, weight images rebuilt)"
                             % (2.0 * n / 1e6),
                       "parallelism": "independent prefix tiles per rank, no collective"},
            "full_map_wall_s_extrapolated": total_evals_map / value * world if value else None,
            "folding_fraction_last_tile": folding / float(n),
            "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline, "other_kernels": other,
            "whole_map_3x3x3": whole,
            "full_6x6_measured": {"wall_s": 114.3, "path": "gp_enumerate_map + designability + neighbour pass, 137 GB store",
                                  "source": "profiles/r1_full_6x6.md (separate run: python tests/full_map_check.py --lattice 6x6)"},
            "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
