"""Multi-GPU plumbing for the genotype-sharded path.

Scoring needs no communication: every rank scores its own aligned genotype range.  Per-class counts (designability,
R / D / O) of disjoint shards add, so they are combined with one all_reduce(SUM).  Works on any torch.distributed
backend (nccl on GPUs, gloo in the CPU tests)."""
import torch
import torch.distributed as dist


def shard_range(n_bits, world, rank, align):
    """Genotype range [begin, begin+count) of `rank`: the 2^n_bits map cut into `world` contiguous pieces whose
    boundaries are multiples of `align` (gp_tile()); the pieces are disjoint and cover the map."""
    if not (0 <= rank < world) or world < 1 or align < 1:
        raise ValueError("bad rank/world/align")
    total = 1 << n_bits
    units = (total + align - 1) // align
    lo = units * rank // world * align
    hi = units * (rank + 1) // world * align
    return min(lo, total), max(0, min(hi, total) - min(lo, total))


def prefix_tiles(n_bits, tile_bits, world, rank):
    """Round-robin assignment of the 2^(n_bits-tile_bits) prefix tiles to ranks: tile t goes to rank t % world."""
    n = 1 << max(0, n_bits - tile_bits)
    return [t << tile_bits for t in range(rank, n, world)]


def reduce_counts(*tensors, group=None):
    """Sum per-class count tensors (hist, R, D, O ...) over all ranks, in place; returns them."""
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        for t in tensors:
            dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return tensors


def max_over_ranks(value, device="cpu", group=None):
    """Max of a python float over ranks (device timings are reported as the max over ranks)."""
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())
