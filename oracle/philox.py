"""Philox4x32-10 counter-based generator (Salmon et al. 2011, "Parallel random numbers: as easy
as 1, 2, 3"), restated in numpy.  The sampler's random draws are defined as functions of
(seed, chain, iteration, draw index) (reading N10), so the GPU path and this oracle
implement the same generator independently.  Pinned by the Random123 known-answer vectors in
tests/golden/philox4x32_10_kat.txt.
"""
import numpy as np

M0 = np.uint64(0xD2511F53)
M1 = np.uint64(0xCD9E8D57)
W0 = np.uint32(0x9E3779B9)
W1 = np.uint32(0xBB67AE85)
MASK = np.uint64(0xFFFFFFFF)


def philox4x32_10(ctr, key):
    """ctr: uint32 [..., 4]; key: uint32 [..., 2] (broadcastable). Returns uint32 [..., 4]."""
    ctr = np.asarray(ctr, dtype=np.uint32)
    key = np.asarray(key, dtype=np.uint32)
    c0, c1, c2, c3 = (ctr[..., i].astype(np.uint64) for i in range(4))
    k0 = np.broadcast_to(key[..., 0], c0.shape).astype(np.uint32)
    k1 = np.broadcast_to(key[..., 1], c0.shape).astype(np.uint32)
    for r in range(10):
        p0 = M0 * c0            # 64-bit products of 32-bit values
        p1 = M1 * c2
        hi0, lo0 = p0 >> np.uint64(32), p0 & MASK
        hi1, lo1 = p1 >> np.uint64(32), p1 & MASK
        n0 = hi1 ^ c1 ^ k0.astype(np.uint64)
        n1 = lo1
        n2 = hi0 ^ c3 ^ k1.astype(np.uint64)
        n3 = lo0
        c0, c1, c2, c3 = n0 & MASK, n1 & MASK, n2 & MASK, n3 & MASK
        with np.errstate(over="ignore"):
            k0 = (k0 + W0).astype(np.uint32)
            k1 = (k1 + W1).astype(np.uint32)
    return np.stack([c0, c1, c2, c3], axis=-1).astype(np.uint32)


def u01(x):
    """uint32 -> double in the open interval (0,1): (x + 0.5) / 2^32."""
    return (np.asarray(x, dtype=np.float64) + 0.5) * (1.0 / 4294967296.0)


def box_muller(x0, x1):
    """two uint32 words -> two independent N(0,1) doubles."""
    r = np.sqrt(-2.0 * np.log(u01(x0)))
    t = 2.0 * np.pi * u01(x1)
    return r * np.cos(t), r * np.sin(t)


class Stream:
    """Draws for one (seed, chain, iteration): word block j is philox(ctr=(j, chain, iteration, tag), key=seed)."""

    def __init__(self, seed, chain, iteration, tag=0):
        self.key = np.array([seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF], dtype=np.uint32)
        self.chain, self.iteration, self.tag = int(chain), int(iteration), int(tag)
        self.j = 0

    def words(self):
        """word block j (blocks are generated 64 at a time; the sequence is the same as one by one)."""
        if self.j % 64 == 0:
            js = (self.j + np.arange(64)) & 0xFFFFFFFF
            ctr = np.empty((64, 4), dtype=np.uint32)
            ctr[:, 0], ctr[:, 1], ctr[:, 2], ctr[:, 3] = js, self.chain, self.iteration, self.tag
            self._buf = philox4x32_10(ctr, self.key)
        out = self._buf[self.j % 64]
        self.j += 1
        return out

    def uniform(self):
        return float(u01(self.words()[0]))

    def normals(self, n):
        out = []
        while len(out) < n:
            w = self.words()
            a, b = box_muller(w[0], w[1])
            c, d = box_muller(w[2], w[3])
            out.extend([float(a), float(b), float(c), float(d)])
        return np.array(out[:n])
