"""Numpy stand-in for libgpmap's reduction calls, with the call names paper_2008_05612_b200/sharding.py uses, so that the
multi-rank orchestration can be driven on CPU under gloo (no GPU here).  Test infrastructure only: it restates the
neighbour-count definition of PAPER.md:138-147 for a shard and for a cross-shard flip."""
import numpy as np
import torch

NULLP = 0xFFFF


class NumpyOps:
    def zeros(self, shape, dtype, like):
        return torch.zeros(shape, dtype=dtype)

    def _np(self, t):
        return t.numpy().view(np.uint16) if t.dtype in (torch.int16, torch.uint16) else t.numpy()

    def designability(self, shard, n_classes):
        s = self._np(shard)
        hist = np.zeros(n_classes + 1, np.int64)
        hist[:n_classes] = np.bincount(s[s != NULLP], minlength=n_classes)
        hist[n_classes] = int((s == NULLP).sum())
        return torch.from_numpy(hist)

    def pair_bitmap(self, n_classes, like):
        return torch.zeros((n_classes * n_classes + 31) // 32, dtype=torch.int32)

    def _count(self, p, q, n_classes, rdo, bitmap):
        live = p != NULLP
        r, d, o = rdo[0].numpy(), rdo[1].numpy(), rdo[2].numpy()
        np.add.at(r, p[live & (q == p)], 1)
        np.add.at(d, p[live & (q == NULLP)], 1)
        other = live & (q != p) & (q != NULLP)
        np.add.at(o, p[other], 1)
        if bitmap is not None and other.any():
            lo = np.minimum(p[other], q[other]).astype(np.int64)
            hi = np.maximum(p[other], q[other]).astype(np.int64)
            bits = np.unique(lo * n_classes + hi)
            w = bitmap.numpy().view(np.uint32)
            np.bitwise_or.at(w, bits >> 5, (np.uint32(1) << (bits & 31).astype(np.uint32)))

    def robustness_partial(self, shard, n_bits, n_classes, rdo, bitmap):
        s = self._np(shard)
        idx = np.arange(s.size)
        for k in range(n_bits):
            self._count(s, s[idx ^ (1 << k)], n_classes, rdo, bitmap)

    def robustness_cross(self, mine, partner, n_classes, rdo, bitmap):
        self._count(self._np(mine), self._np(partner), n_classes, rdo, bitmap)

    def pair_bitmap_or(self, dst, src, n_classes):
        dst |= src

    def pair_bitmap_count(self, bitmap, n_classes):
        return int(np.unpackbits(bitmap.numpy().view(np.uint8)).sum())
