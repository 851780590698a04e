"""Whole GP map of one lattice on one GPU: phenotype store in HBM, designability, neighbour counts, pair count.

    python -m paper_2008_05612_b200.full_map --lattice 6x6 --out gpurun_out/map_6x6

Scores all 2^N genotypes in chunks (progress lines go to <out>/progress.log), then runs gp_designability and
gp_robustness over the resident store and checks the invariants that need no reference:
sum(hist) = 2^N, sum(R+D+O) = N x folding, sum R and sum O even, pheno(rev g) = pheno(g) on a seeded sample.
Writes summary.json and counts.npz (hist, R, D, O).  6x6 needs 137.4 GB for the store (BASELINE.json configs[3])."""
import argparse
import json
import os
import time

import numpy as np

LATTICES = {"4x4": (4, 4, 1), "5x5": (5, 5, 1), "3x3x3": (3, 3, 3), "6x6": (6, 6, 1)}


def bit_reverse(g, n):
    r = np.zeros_like(g)
    for i in range(n):
        r |= ((g >> np.uint64(i)) & np.uint64(1)) << np.uint64(n - 1 - i)
    return r


def run(lattice, out, chunk_bits=30, sample=1 << 20, seed=200805612, keep_store=False, prefix_path=False):
    import torch
    from . import gpmap

    os.makedirs(out, exist_ok=True)
    log = open(os.path.join(out, "progress.log"), "w")

    def say(msg):
        log.write("%.1f %s\n" % (time.time(), msg))
        log.flush()

    S = gpmap.Structures(*LATTICES[lattice])
    N, D, C = S.N, S.D, S.C
    total = 1 << N
    chunk = min(total, 1 << chunk_bits)
    say("lattice %s N=%d D=%d C=%d store %.1f GB" % (lattice, N, D, C, 2.0 * total / 1e9))
    pheno = torch.empty(total, dtype=torch.uint16, device="cuda")
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
    torch.cuda.synchronize()
    ev[0].record()
    if prefix_path:   # gp_enumerate on consecutive ranges: every genotype on all D directed structures
        for b in range(0, total, chunk):
            S.enumerate(b, chunk, pheno[b:b + chunk])
            if (b // chunk) % 8 == 7:
                torch.cuda.synchronize()
                say("scored %d / %d chunks" % (b // chunk + 1, total // chunk))
    else:             # gp_enumerate_map: reversal identity, one representative per class (C columns)
        S.enumerate_map(pheno)
    ev[1].record()
    hist = gpmap.designability(pheno, C)
    ev[2].record()
    R, Dl, Oc, pairs = gpmap.robustness(pheno, N, C)
    ev[3].record()
    torch.cuda.synchronize()
    t_score, t_hist, t_rob = (ev[i].elapsed_time(ev[i + 1]) * 1e-3 for i in range(3))
    say("scoring %.1f s, designability %.2f s, neighbour pass %.1f s" % (t_score, t_hist, t_rob))

    hist = hist.cpu().numpy().astype(np.uint64)
    R, Dl, Oc = (x.cpu().numpy().astype(np.uint64) for x in (R, Dl, Oc))
    folding = int(hist[:C].sum())
    rng = np.random.default_rng(seed)
    g = rng.integers(0, total, size=min(sample, total), dtype=np.uint64)
    gi = torch.from_numpy(g.astype(np.int64)).cuda()
    ri = torch.from_numpy(bit_reverse(g, N).astype(np.int64)).cuda()
    store16 = pheno.view(torch.int16)
    rev_mismatch = int((store16[gi] != store16[ri]).sum().item())
    checks = {
        "hist_sums_to_2^N": int(hist.sum()) == total,
        "R+D+O_equals_N_x_folding": int(R.sum() + Dl.sum() + Oc.sum()) == N * folding,
        "sum_R_even": int(R.sum()) % 2 == 0,
        "sum_O_even": int(Oc.sum()) % 2 == 0,
        "reversal_symmetry_sample_mismatches": rev_mismatch,
    }
    order = np.argsort(hist[:C])[::-1]
    summary = {
        "lattice": lattice, "N": N, "D": D, "C": C, "genotypes": total, "evaluations": float(total) * D,
        "path": "gp_enumerate (prefix tiles, D columns)" if prefix_path else "gp_enumerate_map (reversal identity, C columns)",
        "evaluations_executed": float(total) * (D if prefix_path else C),
        "seconds": {"scoring": t_score, "designability": t_hist, "neighbour_pass": t_rob,
                    "total": t_score + t_hist + t_rob},
        "evals_per_s_scoring": float(total) * D / t_score,
        "folding": folding, "folding_fraction": folding / total, "null": int(hist[C]),
        "designable_classes": int((hist[:C] > 0).sum()), "top5_designability": [int(hist[i]) for i in order[:5]],
        "sum_R": int(R.sum()), "sum_D": int(Dl.sum()), "sum_O": int(Oc.sum()), "phenotype_pairs": int(pairs.item()),
        "isolated_designable_classes": int(((Oc == 0) & (hist[:C] > 0)).sum()),
        "checks": checks,
    }
    np.savez_compressed(os.path.join(out, "counts.npz"), hist=hist, R=R, D=Dl, O=Oc)
    with open(os.path.join(out, "summary.json"), "w") as f:
        json.dump(summary, f, indent=1)
    say("done " + json.dumps(checks))
    log.close()
    return (summary, pheno, S) if keep_store else summary


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--lattice", default="6x6", choices=sorted(LATTICES))
    ap.add_argument("--out", default="gpurun_out/map")
    ap.add_argument("--chunk-bits", type=int, default=30)
    ap.add_argument("--prefix-path", action="store_true", help="score with gp_enumerate instead of gp_enumerate_map")
    a = ap.parse_args()
    print(json.dumps(run(a.lattice, a.out, a.chunk_bits, prefix_path=a.prefix_path)))


if __name__ == "__main__":
    main()
