"""Not collected by pytest (long): full-map run of one lattice on the GPU + oracle parity on sampled genotype ranges.

    python tests/full_map_check.py --lattice 6x6 --out gpurun_out/map_6x6 --ranges 8 --length 2048

Runs paper_2008_05612_b200.full_map (whole store resident in HBM), then compares `ranges` ranges of `length`
consecutive phenotypes (first, last, seeded-random: workloads.sample_ranges) element by element with the CPU oracle,
and, for maps the oracle can finish (N <= 25), the whole histogram / R / D / O / pair count."""
import argparse
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import workloads  # noqa: E402
from oracle import gp_oracle as orc  # noqa: E402
from paper_2008_05612_b200 import full_map  # noqa: E402


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--lattice", default="6x6")
    ap.add_argument("--out", default="gpurun_out/map")
    ap.add_argument("--ranges", type=int, default=8)
    ap.add_argument("--length", type=int, default=2048)
    ap.add_argument("--prefix-path", action="store_true")
    a = ap.parse_args()
    summary, pheno, S = full_map.run(a.lattice, a.out, keep_store=True, prefix_path=a.prefix_path)
    O = orc.Structures(*full_map.LATTICES[a.lattice])
    bad = 0
    for b, c in workloads.sample_ranges(S.N, a.ranges, a.length, 512):
        got = pheno[b:b + c].cpu().numpy()
        want = O.enumerate(b, c, want_gap=False)
        bad += int((got != want).sum())
    verdict = {"sampled_ranges": a.ranges, "range_length": a.length, "sampled_mismatches_vs_oracle": bad}
    if S.N <= 25:
        store = pheno.cpu().numpy()
        whole = O.enumerate(0, 1 << S.N, want_gap=False)
        Ro, Do, Oo, pco = orc.robustness(whole, S.N, S.C)
        cnt = np.load(os.path.join(a.out, "counts.npz"))
        verdict["whole_map_equal"] = bool(np.array_equal(store, whole) and np.array_equal(cnt["R"], Ro)
                                          and np.array_equal(cnt["D"], Do) and np.array_equal(cnt["O"], Oo)
                                          and summary["phenotype_pairs"] == pco
                                          and np.array_equal(cnt["hist"], orc.designability(whole, S.C)))
    summary["oracle_parity"] = verdict
    with open(os.path.join(a.out, "summary.json"), "w") as f:
        json.dump(summary, f, indent=1)
    print(json.dumps(summary))
    ok = bad == 0 and all(v is True or v == 0 for v in summary["checks"].values()) and verdict.get("whole_map_equal", True)
    sys.exit(0 if ok else 1)


if __name__ == "__main__":
    main()
