"""Whole GP map of one lattice on one GPU, in resumable pieces: phenotype store in HBM, designability, neighbour counts,
pair count.

    python -m paper_2008_05612_b200.full_map --lattice 6x6 --out gpurun_out/map_6x6 [--chunks 64]
    python -m paper_2008_05612_b200.full_map --lattice 3x3x3 --out out/map_333 --checkpoint-store [--resume]
    torchrun --nproc-per-node 8 -m paper_2008_05612_b200.full_map --lattice 6x6 --out out/map_6x6 --sharded

The map is scored as `chunks` ranges of units through gp_enumerate_map_range (include/gpmap.h; the paper's own 110-day
job survived by appending results run by run).  After every chunk <out>/progress.json
records the units done; with --checkpoint-store the store is also saved (<out>/store.u16, sensible up to 3x3x3), and
--resume continues from the recorded chunk instead of starting over; --resume without a saved store (or with other
settings than the interrupted run) is an error, never a silent restart.  Then gp_reduce_store runs over the resident
store and the invariants that need no reference are checked: sum(hist) = 2^N,
sum(R+D+O) = N x folding, sum R and sum O even, pheno(rev g) = pheno(g) on a seeded sample, and gp_phi_row of the most
and least designable class against R / D / O of the tiled neighbour pass
(tests/test_gpu_map_range.py::test_full_map_run_survives_an_interruption compares such a run with the CPU oracle).
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


def phi_row_witness(gpmap, pheno, n_bits, C, hist, R, Dl, Oc):
    """An independent witness for the tiled neighbour pass on stores the oracle cannot reach (the 6x6 map's third pass):
    gp_phi_row — another, untiled kernel — for the most designable class and the rarest non-empty one.  Adjacency is
    symmetric, so with row[p] = flips leading from class p into q (Eq. 2 numerators):
    row[q] = R[q], sum_{p != q} row[p] = O[q], row[C] (from null genotypes) = D[q].  Returns {check name: bool}."""
    designable = np.nonzero(hist[:C])[0]
    if designable.size == 0:
        return {}
    top = int(designable[np.argmax(hist[designable])])
    rare = int(designable[np.argmin(hist[designable])])
    out = {}
    for name, q in (("top", top), ("rarest", rare)):
        row = gpmap.phi_row(pheno, n_bits, C, q).cpu().numpy().astype(np.uint64)
        out["phi_row_%s_equals_R" % name] = int(row[q]) == int(R[q])
        out["phi_row_%s_sums_to_O" % name] = int(row[:C].sum() - row[q]) == int(Oc[q])
        out["phi_row_%s_from_null_equals_D" % name] = int(row[C]) == int(Dl[q])
    return out


def run(lattice, out, chunks=64, sample=1 << 20, seed=200805612, keep_store=False, prefix_path=False, resume=False,
        checkpoint_store=False, stop_after=None):
    """stop_after = number of chunks after which the run stops as if interrupted (returns None); used by the tests."""
    import torch
    from . import gpmap

    os.makedirs(out, exist_ok=True)
    prog_path, store_path = os.path.join(out, "progress.json"), os.path.join(out, "store.u16")
    S = gpmap.Structures(*LATTICES[lattice])
    N, D, C = S.N, S.D, S.C
    total = 1 << N
    U = S.map_units()
    chunks = max(1, min(chunks, U))
    done_chunks, seconds_before = 0, 0.0
    if resume:   # never restart silently: a resume that cannot continue is an error the caller must see
        if not os.path.exists(prog_path):
            raise RuntimeError("--resume: %s does not exist; start the run without --resume" % prog_path)
        with open(prog_path) as f:
            prog = json.load(f)
        same = (prog.get("lattice"), prog.get("chunks"), prog.get("units"), prog.get("prefix_path")) == (lattice, chunks, U, prefix_path)
        if not same:
            raise RuntimeError("--resume: %s was written by a run with other settings (lattice / chunks / units / path): %r"
                               % (prog_path, prog))
        if not (prog.get("store_saved") and os.path.exists(store_path)):
            raise RuntimeError("--resume: the interrupted run saved no store (%s); only a run started with "
                               "--checkpoint-store can be resumed" % store_path)
        done_chunks, seconds_before = prog["chunks_done"], prog.get("scoring_seconds", 0.0)
    pheno = torch.empty(total, dtype=torch.uint16, device="cuda")
    if done_chunks:
        pheno.copy_(torch.from_numpy(np.fromfile(store_path, dtype=np.int16)).view(torch.uint16))
    log = open(os.path.join(out, "progress.log"), "a" if done_chunks else "w")

    def say(msg):
        log.write("%.1f %s\n" % (time.time(), msg))
        log.flush()

    say("lattice %s N=%d D=%d C=%d units=%d store %.1f GB, starting at chunk %d of %d" % (lattice, N, D, C, U, 2.0 * total / 1e9,
                                                                                         done_chunks, chunks))
    t_score = seconds_before
    for c in range(done_chunks, chunks):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        if prefix_path:   # gp_enumerate on consecutive ranges: every genotype on all D directed structures
            b0, b1 = total * c // chunks // 512 * 512, (total * (c + 1) // chunks // 512 * 512 if c + 1 < chunks else total)
            S.enumerate(b0, b1 - b0, pheno[b0:b1])
        else:             # reversal identity, one representative per class (C columns)
            u0, u1 = U * c // chunks, U * (c + 1) // chunks
            S.enumerate_map_range(u0, u1 - u0, pheno)
        e1.record()
        torch.cuda.synchronize()
        t_score += e0.elapsed_time(e1) * 1e-3
        prog = {"lattice": lattice, "chunks": chunks, "units": U, "prefix_path": prefix_path, "chunks_done": c + 1,
                "scoring_seconds": t_score, "store_saved": False}
        if checkpoint_store:
            pheno.view(torch.int16).cpu().numpy().tofile(store_path + ".tmp")
            os.replace(store_path + ".tmp", store_path)
            prog["store_saved"] = True
        with open(prog_path + ".tmp", "w") as f:
            json.dump(prog, f)
        os.replace(prog_path + ".tmp", prog_path)
        if (c + 1) % 8 == 0 or c + 1 == chunks:
            say("scored %d / %d chunks, %.1f s" % (c + 1, chunks, t_score))
        if stop_after is not None and c + 1 - done_chunks >= stop_after and c + 1 < chunks:
            say("stopped after %d chunks (as if interrupted)" % (c + 1))
            log.close()
            S.close()
            return None
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    ev[0].record()
    hist, R, Dl, Oc, pairs = gpmap.reduce_store(pheno, N, C)   # designability comes out of the neighbour pass's first sweep
    ev[1].record()
    torch.cuda.synchronize()
    t_red = ev[0].elapsed_time(ev[1]) * 1e-3
    say("scoring %.1f s, designability + neighbour pass %.2f s" % (t_score, t_red))

    hist = hist.cpu().numpy().astype(np.uint64)
    R, Dl, Oc = (x.cpu().numpy().astype(np.uint64) for x in (R, Dl, Oc))
    folding = int(hist[:C].sum())
    witness = phi_row_witness(gpmap, pheno, N, C, hist, R, Dl, Oc)
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
    checks.update(witness)
    order = np.argsort(hist[:C])[::-1]
    summary = {
        "lattice": lattice, "N": N, "D": D, "C": C, "genotypes": total, "evaluations": float(total) * D,
        "path": "gp_enumerate (prefix tiles, D columns)" if prefix_path else "gp_enumerate_map_range (reversal identity, C columns)",
        "chunks": chunks, "resumed_at_chunk": done_chunks,
        "evaluations_executed": float(total) * (D if prefix_path else C),
        "seconds": {"scoring": t_score, "designability_and_neighbour_pass": t_red, "total": t_score + t_red},
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


def run_sharded(lattice, out, backend=None):
    """Whole map over the ranks of a torch.distributed job (torchrun, one process per GPU): the store is sharded on the
    top log2(world) genotype bits (sharding.py).  Every rank scores its own shard with gp_enumerate,
    reduces it with libgpmap and exchanges shards / counts / pair bitmap; rank 0 writes summary.json.  With 8 GPUs the
    6x6 store is 17 GB per rank."""
    import torch
    import torch.distributed as dist
    from . import gpmap, sharding

    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local % max(1, torch.cuda.device_count()))
    if not dist.is_initialized():
        dist.init_process_group(backend or ("nccl" if torch.cuda.device_count() >= world else "gloo"))
    S = gpmap.Structures(*LATTICES[lattice])
    N, D, C = S.N, S.D, S.C
    b, c = sharding.shard_range(N, world, rank, gpmap.tile())
    shard = torch.empty(c, dtype=torch.uint16, device="cuda")
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    dist.barrier()
    torch.cuda.synchronize()
    ev[0].record()
    step = 1 << 30
    for off in range(0, c, step):
        S.enumerate(b + off, min(step, c - off), shard[off:off + step])
    ev[1].record()
    comm = sharding.DistComm()
    hist, R, Dl, Oc, pairs = sharding.reduce_store_sharded(sharding.LibOps(), comm, shard, N, C)
    ev[2].record()
    torch.cuda.synchronize()
    dev = "cpu" if comm.backend == "gloo" else "cuda"
    t_score = comm.max_(ev[0].elapsed_time(ev[1]) * 1e-3, dev)
    t_red = comm.max_(ev[1].elapsed_time(ev[2]) * 1e-3, dev)
    summary = None
    if rank == 0:
        hist = hist.cpu().numpy().astype(np.uint64)
        R, Dl, Oc = (x.cpu().numpy().astype(np.uint64) for x in (R, Dl, Oc))
        folding = int(hist[:C].sum())
        summary = {"lattice": lattice, "N": N, "D": D, "C": C, "world": world, "genotypes": 1 << N,
                   "path": "gp_enumerate per rank (prefix tiles, D columns), sharded reductions",
                   "seconds": {"scoring": t_score, "reductions_and_exchange": t_red, "total": t_score + t_red},
                   "evals_per_s_scoring": float(1 << N) * D / t_score,
                   "bytes_sent_per_rank": comm.bytes_sent, "folding": folding, "null": int(hist[C]),
                   "sum_R": int(R.sum()), "sum_D": int(Dl.sum()), "sum_O": int(Oc.sum()), "phenotype_pairs": int(pairs),
                   "checks": {"hist_sums_to_2^N": int(hist.sum()) == 1 << N,
                              "R+D+O_equals_N_x_folding": int(R.sum() + Dl.sum() + Oc.sum()) == N * folding,
                              "sum_R_even": int(R.sum()) % 2 == 0, "sum_O_even": int(Oc.sum()) % 2 == 0}}
        os.makedirs(out, exist_ok=True)
        np.savez_compressed(os.path.join(out, "counts.npz"), hist=hist, R=R, D=Dl, O=Oc)
        with open(os.path.join(out, "summary.json"), "w") as f:
            json.dump(summary, f, indent=1)
    dist.barrier()
    S.close()
    dist.destroy_process_group()
    return summary


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--lattice", default="6x6", choices=sorted(LATTICES))
    ap.add_argument("--out", default="gpurun_out/map")
    ap.add_argument("--chunks", type=int, default=64)
    ap.add_argument("--resume", action="store_true", help="continue from <out>/progress.json (needs a saved store)")
    ap.add_argument("--checkpoint-store", action="store_true", help="save the store after every chunk (up to 3x3x3)")
    ap.add_argument("--prefix-path", action="store_true", help="score with gp_enumerate instead of gp_enumerate_map_range")
    ap.add_argument("--sharded", action="store_true", help="run under torchrun: the store sharded over the ranks (sharding.py)")
    a = ap.parse_args()
    if a.sharded:
        summary = run_sharded(a.lattice, a.out)
        if summary is not None:
            print(json.dumps(summary))
        raise SystemExit(0 if summary is None or all(summary["checks"].values()) else 1)
    summary = run(a.lattice, a.out, a.chunks, prefix_path=a.prefix_path, resume=a.resume, checkpoint_store=a.checkpoint_store)
    print(json.dumps(summary))
    raise SystemExit(0 if all(v is True or v == 0 for v in summary["checks"].values()) else 1)


if __name__ == "__main__":
    main()
