"""Multi-GPU orchestration of the hot path ("a network of GPUs").

The phenotype store of a 2^n_bits sub-cube is sharded over `world` = 2^q ranks on its TOP q genotype bits: rank r owns
genotypes [r * 2^(n_bits-q), (r+1) * 2^(n_bits-q)).  One process per GPU.

  scoring        rank-local: gp_enumerate on the rank's own range, no communication;
  designability  rank-local histogram, then all_reduce(SUM);
  neighbour pass flips of the n_bits-q low bits are rank-local (gp_robustness_partial on the shard); the flip of top bit
                 b pairs rank r with rank r ^ 2^b: the two ranks swap their shards (one send + one receive of
                 2^(n_bits-q+1) bytes per rank and bit — a hypercube exchange — in chunks, so the receive buffer stays
                 small) and each runs gp_robustness_cross(mine, partner's); R / D / O all_reduce(SUM);
  pair bitmap    every rank ORs its own events into a private bitmap; the bitmaps are OR-reduced (gloo: all_reduce(BOR);
                 NCCL has no bitwise reduction, so ranks all_gather the bitmaps and gp_pair_bitmap_or them locally);
  components     not sharded ("replicas only").

Every kernel call goes through an `ops` object with libgpmap's call names (LibOps below binds them to gpmap.py); the
communication goes through torch.distributed (NcclComm / GlooComm) or, for single-process tests that play all ranks
one after the other on one device, PeerComm, where "exchange" is a peer pointer — the NVLink peer-load variant of the
same step.  tests/test_sharding_gloo.py drives this module with world_size 2 on CPU; tests/test_gpu_sharding.py drives
it with libgpmap for 2 and 4 emulated ranks and compares with the single-rank result."""
import torch
import torch.distributed as dist


def log2_exact(world):
    q = world.bit_length() - 1
    if world < 1 or (1 << q) != world:
        raise ValueError("world size must be a power of two to shard on genotype bits")
    return q


def shard_range(n_bits, world, rank, align=1):
    """Genotype range [begin, begin+count) of `rank`: the 2^n_bits map cut into `world` contiguous pieces whose
    boundaries are multiples of `align` (gp_tile()); the pieces are disjoint and cover the map."""
    if not (0 <= rank < world) or world < 1 or align < 1:
        raise ValueError("bad rank/world/align")
    total = 1 << n_bits
    units = (total + align - 1) // align
    lo = units * rank // world * align
    hi = units * (rank + 1) // world * align
    return min(lo, total), max(0, min(hi, total) - min(lo, total))


class LibOps:
    """libgpmap's reductions on CUDA tensors (argument marshalling only)."""

    def __init__(self):
        from . import gpmap
        self.g = gpmap

    def zeros(self, shape, dtype, like):
        return torch.zeros(shape, dtype=dtype, device=like.device)

    def designability(self, shard, n_classes):
        return self.g.designability(shard, n_classes)

    def pair_bitmap(self, n_classes, like):
        return self.g.pair_bitmap(n_classes, device=like.device)

    def robustness_partial(self, shard, n_bits, n_classes, rdo, bitmap):
        self.g.robustness_partial(shard, n_bits, n_classes, rdo, bitmap)

    def robustness_cross(self, mine, partner, n_classes, rdo, bitmap):
        self.g.robustness_cross(mine, partner, n_classes, rdo, bitmap)

    def pair_bitmap_or(self, dst, src, n_classes):
        self.g.pair_bitmap_or(dst, src, n_classes)

    def pair_bitmap_count(self, bitmap, n_classes):
        return self.g.pair_bitmap_count(bitmap, n_classes)   # device tensor: no host synchronisation on the path


class DistComm:
    """torch.distributed plumbing: NCCL between GPUs, gloo in the CPU tests (same calls)."""

    def __init__(self, group=None):
        self.group = group
        self.rank = dist.get_rank(group)
        self.world = dist.get_world_size(group)
        self.backend = dist.get_backend(group)
        self.bytes_sent = 0

    def exchange(self, mine, partner_rank, chunk, offset):
        """Swap `chunk` entries at `offset` of the shard with the partner rank; returns the partner's entries."""
        send = mine[offset:offset + chunk]
        stage = self.backend == "gloo" and send.is_cuda     # gloo moves host memory only: stage device shards through it
        src = send.cpu() if stage else send
        recv = torch.empty_like(src)
        # 16-bit integers are not an NCCL data type: ship the bytes
        ops = [dist.P2POp(dist.isend, src.view(torch.uint8), partner_rank, self.group),
               dist.P2POp(dist.irecv, recv.view(torch.uint8), partner_rank, self.group)]
        for req in dist.batch_isend_irecv(ops):
            req.wait()
        self.bytes_sent += send.numel() * send.element_size()
        return recv.to(send.device) if stage else recv

    def sum_(self, *tensors):
        for t in tensors:
            if self.backend == "gloo" and t.is_cuda:
                h = t.cpu()
                dist.all_reduce(h, op=dist.ReduceOp.SUM, group=self.group)
                t.copy_(h)
            else:
                dist.all_reduce(t, op=dist.ReduceOp.SUM, group=self.group)
            self.bytes_sent += t.numel() * t.element_size()
        return tensors

    def or_(self, bitmap, ops, n_classes):
        """OR-reduce the pair bitmaps of all ranks, in place."""
        if self.world == 1:
            return bitmap
        if self.backend == "gloo":
            h = bitmap.cpu() if bitmap.is_cuda else bitmap
            dist.all_reduce(h, op=dist.ReduceOp.BOR, group=self.group)
            if bitmap.is_cuda:
                bitmap.copy_(h)
        else:
            parts = [torch.empty_like(bitmap) for _ in range(self.world)]
            dist.all_gather(parts, bitmap, group=self.group)
            for r, p in enumerate(parts):
                if r != self.rank:
                    ops.pair_bitmap_or(bitmap, p, n_classes)
        self.bytes_sent += bitmap.numel() * bitmap.element_size()
        return bitmap

    def max_(self, value, device="cpu"):
        t = torch.tensor([float(value)], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX, group=self.group)
        return float(t.item())


class PeerComm:
    """All shards live in one process (tests on one device; or one process driving peer-mapped GPUs): the partner's
    shard is read in place — the peer-load variant of the exchange.  Reductions are done by `combine_partials`."""

    def __init__(self, shards, rank):
        self.shards, self.rank, self.world, self.bytes_sent = shards, rank, len(shards), 0

    def exchange(self, mine, partner_rank, chunk, offset):
        self.bytes_sent += chunk * mine.element_size()
        return self.shards[partner_rank][offset:offset + chunk]


def local_part(ops, comm, shard, n_bits, n_classes, chunk_entries=1 << 29):
    """One rank's share of a5 + a6 over the sharded 2^n_bits store: (hist, rdo[3, C], bitmap), before reduction."""
    q = log2_exact(comm.world)
    local_bits = n_bits - q
    if shard.numel() != 1 << local_bits:
        raise ValueError("shard must hold 2^(n_bits - log2 world) entries")
    hist = ops.designability(shard, n_classes)
    rdo = ops.zeros((3, n_classes), torch.int64, shard)
    bitmap = ops.pair_bitmap(n_classes, shard)
    if local_bits >= 1:
        ops.robustness_partial(shard, local_bits, n_classes, rdo, bitmap)
    for b in range(q):                                   # flips of the rank-selecting bits: hypercube exchange
        partner = comm.rank ^ (1 << b)
        for off in range(0, shard.numel(), chunk_entries):
            cnt = min(chunk_entries, shard.numel() - off)
            theirs = comm.exchange(shard, partner, cnt, off)
            ops.robustness_cross(shard[off:off + cnt], theirs, n_classes, rdo, bitmap)
    return hist, rdo, bitmap


def reduce_store_sharded(ops, comm, shard, n_bits, n_classes, chunk_entries=1 << 29):
    """a5 + a6 of the whole sharded store on every rank: (hist, R, D, O, pair_count), identical on all ranks and
    identical to gp_designability + gp_robustness over the unsharded store."""
    hist, rdo, bitmap = local_part(ops, comm, shard, n_bits, n_classes, chunk_entries)
    comm.sum_(hist, rdo)
    comm.or_(bitmap, ops, n_classes)
    return hist, rdo[0], rdo[1], rdo[2], ops.pair_bitmap_count(bitmap, n_classes)


def combine_partials(ops, partials, n_classes):
    """Reduction of the per-rank partial results when one process holds them all (PeerComm)."""
    hist = partials[0][0].clone()
    rdo = partials[0][1].clone()
    bitmap = partials[0][2].clone()
    for h, r, b in partials[1:]:
        hist += h
        rdo += r
        ops.pair_bitmap_or(bitmap, b, n_classes)
    return hist, rdo[0], rdo[1], rdo[2], ops.pair_bitmap_count(bitmap, n_classes)


def exchange_bytes_per_rank(n_bits, world, n_classes):
    """Bytes one rank sends for a5 + a6 of a 2^n_bits store: q shard swaps, four count vectors,
    one pair bitmap."""
    q = log2_exact(world)
    return q * (2 << (n_bits - q)) + 8 * (4 * n_classes + 1) + 4 * ((n_classes * n_classes + 31) // 32)
