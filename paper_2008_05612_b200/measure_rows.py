"""Time every row of the hot path on the configuration BASELINE.json names for it.

    python -m paper_2008_05612_b200.measure_rows [--out gpurun_out/rows.json]

Device times are CUDA-event times on the launching stream after one warm-up call; a0 is host wall time."""
import argparse
import json
import time

import torch

from . import gpmap

SEED = 200805612


def dev_time(fn, reps=2):
    fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        out = fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) * 1e-3 / reps, out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default="gpurun_out/rows.json")
    ap.add_argument("--mj-log2", type=int, default=30)
    a = ap.parse_args()
    rows = []
    structs = {}
    for name, dims in (("4x4", (4, 4, 1)), ("5x5", (5, 5, 1)), ("3x3x3", (3, 3, 3)), ("6x6", (6, 6, 1))):
        t0 = time.perf_counter()
        structs[name] = gpmap.Structures(*dims)
        rows.append(dict(row="a0 gp_structures", config=name, seconds=time.perf_counter() - t0,
                         note="host DFS + canonicalisation + upload, D=%d C=%d" % (structs[name].D, structs[name].C)))
    for name in ("4x4", "5x5", "3x3x3"):
        S = structs[name]
        n = 1 << S.N
        ph = torch.empty(n, dtype=torch.uint16, device="cuda")
        t, _ = dev_time(lambda: S.enumerate(0, n, ph))
        rows.append(dict(row="a1-a4 gp_enumerate (prefix path, D columns)", config=name, seconds=t, evals_per_s=n * S.D / t))
        t, _ = dev_time(lambda: S.enumerate_map(ph))
        rows.append(dict(row="a1-a4 gp_enumerate_map (reversal identity, C columns)", config=name, seconds=t,
                         effective_evals_per_s=n * S.D / t))
        t, _ = dev_time(lambda: S.enumerate(0, min(n, 1 << 22), ph, simple=True), reps=1)
        rows.append(dict(row="a1-a4 gp_enumerate_simple (CUDA cores, like the paper's kernel)", config=name + " first 2^22",
                         seconds=t, evals_per_s=min(n, 1 << 22) * S.D / t))
        t, _ = dev_time(lambda: gpmap.designability(ph, S.C))
        rows.append(dict(row="a5 gp_designability", config=name, seconds=t, GBps=2.0 * n / t / 1e9))
        t, _ = dev_time(lambda: gpmap.robustness(ph, S.N, S.C))
        rows.append(dict(row="a6 gp_robustness (+ pair bitmap)", config=name, seconds=t, GBps_algorithmic=2.0 * n / t / 1e9))
        if S.N <= 27:
            t, _ = dev_time(lambda: gpmap.nn_components(ph, S.N, S.C), reps=1)
            rows.append(dict(row="a7 gp_nn_components", config=name, seconds=t))
        del ph
    # the paper's sampling runs (Table 3): random H/P sequences, each against every fold
    import numpy as np
    for name, paper_s in (("6x6", 1.35e-4), ("3x3x3", 2.6e-4)):
        S = structs[name]
        cnt = 1 << 21
        seqs = torch.from_numpy(np.random.default_rng(SEED).integers(0, 2, size=(cnt, S.N), dtype=np.uint8)).cuda()
        ph = torch.empty(cnt, dtype=torch.uint16, device="cuda")
        e = np.array(gpmap.HP_ENERGIES, np.int32)
        for label, on, c in (("tensor-core sequence_kernel", 1, cnt), ("CUDA-core kernel", 0, 1 << 17)):
            gpmap.lib().gp_set_seq_tc(on)
            t, _ = dev_time(lambda: S.enumerate_seqs(seqs[:c], ph[:c], None, e=e, alphabet=2), reps=1)
            rows.append(dict(row="sampling: gp_enumerate_seqs, random HP sequences (%s)" % label, config="%s, %d sequences" % (name, c),
                             seconds=t, evals_per_s=c * S.D / t, seconds_per_sequence=t / c,
                             paper_gpu_seconds_per_sequence=paper_s))
        gpmap.lib().gp_set_seq_tc(1)
        del seqs, ph
    S = structs["4x4"]
    M = gpmap.seeded_matrix(SEED)
    n = 1 << a.mj_log2
    ph = torch.empty(n, dtype=torch.uint16, device="cuda")
    t, _ = dev_time(lambda: S.enumerate_seeded(SEED, 0, n, ph, e=M), reps=1)
    hist = gpmap.designability(ph, S.C)
    rows.append(dict(row="a8 gp_enumerate_seeded (20 letters, seeded matrix)", config="4x4, 2^%d sequences" % a.mj_log2, seconds=t,
                     evals_per_s=n * S.D / t, folding_fraction=1.0 - hist[S.C].item() / n))
    with open(a.out, "w") as f:
        json.dump(rows, f, indent=1)
    for r in rows:
        print(json.dumps(r))


if __name__ == "__main__":
    main()
