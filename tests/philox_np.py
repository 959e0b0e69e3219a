"""Independent numpy restatement of Philox4x32-10 and of the counter packing of DESIGN.md §3.5.

Used by the tests to re-derive, outside both the oracle and the CUDA path, the random numbers a
given (domain, site, system, counter) consumes.  Vectorised over arrays of counters.
"""
import numpy as np

M0, M1 = np.uint64(0xD2511F53), np.uint64(0xCD9E8D57)
W0, W1 = 0x9E3779B9, 0xBB67AE85
DOMAIN_INIT, DOMAIN_HB, DOMAIN_PT = 0, 1, 2
MASK = np.uint64(0xFFFFFFFF)


def philox4x32_10(c0, c1, c2, c3, k0, k1):
    c0, c1, c2, c3 = (np.asarray(c, dtype=np.uint64) & MASK for c in (c0, c1, c2, c3))
    c0, c1, c2, c3 = np.broadcast_arrays(c0, c1, c2, c3)
    k0 = int(k0) & 0xFFFFFFFF
    k1 = int(k1) & 0xFFFFFFFF
    for r in range(10):
        p0 = M0 * c0
        p1 = M1 * c2
        hi0, lo0 = p0 >> np.uint64(32), p0 & MASK
        hi1, lo1 = p1 >> np.uint64(32), p1 & MASK
        c0, c1, c2, c3 = hi1 ^ c1 ^ np.uint64(k0), lo1, hi0 ^ c3 ^ np.uint64(k1), lo0
        k0 = (k0 + W0) & 0xFFFFFFFF
        k1 = (k1 + W1) & 0xFFFFFFFF
    return tuple(c.astype(np.uint32) for c in (c0, c1, c2, c3))


def u01(w):
    """23-bit midpoint uniform: ((w>>9) + 0.5) * 2^-23, as float64 (exact)."""
    return ((np.asarray(w, dtype=np.uint32) >> np.uint32(9)).astype(np.float64) + 0.5) / 8388608.0


def draw(domain, c0, k, c2, seed):
    """Words of the Philox call for (domain, c0, counter k, c2) under key = seed."""
    k = int(k)
    c1 = k & 0xFFFFFFFF
    c3 = ((k >> 32) & 0x0FFFFFFF) | (domain << 28)
    return philox4x32_10(c0, c1, c2, c3, seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF)
