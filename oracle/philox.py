"""O1 -- Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), test oracle.

The paper says only "a PRNG seeded from /dev/urandom ... compute a random permutation"
(section 5 "Implementation Details"); BJ:north_star fixes the generator:
"cloak_keygen (a Philox4x32-10 keyed permutation, defined as indices sorted by
Philox(key, index))".

One round, on a 128-bit counter (c0,c1,c2,c3) and a 64-bit key (k0,k1), all 32-bit words:
    (hi0, lo0) = 0xD2511F53 * c0        (32x32 -> 64)
    (hi1, lo1) = 0xCD9E8D57 * c2
    (c0, c1, c2, c3) <- (hi1 ^ c1 ^ k0,  lo1,  hi0 ^ c3 ^ k1,  lo0)
and after every round  k0 += 0x9E3779B9,  k1 += 0xBB67AE85  (mod 2^32).
Ten rounds; the key bump after the tenth is unused.
"""
import numpy as np

_M0 = np.uint64(0xD2511F53)
_M1 = np.uint64(0xCD9E8D57)
_W0 = np.uint64(0x9E3779B9)
_W1 = np.uint64(0xBB67AE85)
_LO = np.uint64(0xFFFFFFFF)
_32 = np.uint64(32)


def philox4x32_10(c0, c1, c2, c3, k0, k1):
    """Vectorised over equal-shaped (or broadcastable) arrays of 32-bit words.

    Every argument is anything numpy can turn into uint64 holding a value < 2^32.
    Returns four uint32 arrays (o0, o1, o2, o3).
    """
    c0, c1, c2, c3, k0, k1 = np.broadcast_arrays(
        *[np.asarray(a, dtype=np.uint64) for a in (c0, c1, c2, c3, k0, k1)])
    for a in (c0, c1, c2, c3, k0, k1):
        if a.size and int(a.max()) > 0xFFFFFFFF:
            raise ValueError("philox words must be < 2^32")
    c0, c1, c2, c3, k0, k1 = [a.copy() for a in (c0, c1, c2, c3, k0, k1)]
    for _ in range(10):
        p0 = _M0 * c0                     # < 2^64, exact in uint64
        p1 = _M1 * c2
        hi0, lo0 = p0 >> _32, p0 & _LO
        hi1, lo1 = p1 >> _32, p1 & _LO
        c0, c1, c2, c3 = hi1 ^ c1 ^ k0, lo1, hi0 ^ c3 ^ k1, lo0
        k0 = (k0 + _W0) & _LO
        k1 = (k1 + _W1) & _LO
    return tuple(a.astype(np.uint32) for a in (c0, c1, c2, c3))
