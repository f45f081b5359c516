"""O2 / O3 -- keyed permutation = indices sorted by Philox(key, index).  Test oracle.

BJ:north_star: "cloak_keygen (a Philox4x32-10 keyed permutation, defined as indices sorted by
Philox(key, index))".  Paper: "a random permutation is computed" before any page is allocated
or any weight transferred.  The counter layout, output words, sort direction and
tie-break are silent in both; reading G2 / O2 is used:

    for i in [0, n):  o = Philox(ctr = (i mod 2^32, i >> 32, stream mod 2^32, stream >> 32),
                                 key = (key mod 2^32, key >> 32))
                      r_i = (o[0] << 32) | o[1]
    perm = indices 0..n-1 sorted ascending by the pair (r_i, i);   inv[perm[j]] = j.

Direction (G3): gather form dst[j] = src[perm[j]]; logical item i lives at position inv[i].
"""
import numpy as np
from .philox import philox4x32_10

# O3 stream ids: purpose in the high 32-bit word.
STREAM_BLOCK = 1 << 32
STREAM_PAGE = 2 << 32
STREAM_TENSOR = 3 << 32


def stream_mlp(layer):
    return (4 << 32) | layer


def stream_kvhead(layer):
    return (5 << 32) | layer


def stream_qgroup(layer, n_kv, g):
    return (6 << 32) | (layer * n_kv + g)


def sort_keys(key, stream, n):
    """r_i of O2 for i in [0, n), uint64."""
    if not (1 <= n < 2 ** 32):
        raise ValueError("n must be in [1, 2^32)")
    i = np.arange(n, dtype=np.uint64)
    o0, o1, _, _ = philox4x32_10(i & np.uint64(0xFFFFFFFF), i >> np.uint64(32),
                                 stream & 0xFFFFFFFF, (stream >> 32) & 0xFFFFFFFF,
                                 key & 0xFFFFFFFF, (key >> 32) & 0xFFFFFFFF)
    return (o0.astype(np.uint64) << np.uint64(32)) | o1.astype(np.uint64)


def sort_pairs(r):
    """perm, inv from sort keys r: ascending by (r_i, i).  Separate so ties can be forced."""
    r = np.asarray(r, dtype=np.uint64)
    n = r.shape[0]
    idx = np.arange(n, dtype=np.uint64)
    perm = np.lexsort((idx, r)).astype(np.uint32)      # last key is primary: (r, then i)
    inv = np.empty(n, dtype=np.uint32)
    inv[perm] = np.arange(n, dtype=np.uint32)
    return perm, inv


def keygen(key, stream, n):
    """(perm, inv), each n x uint32 -- O2."""
    return sort_pairs(sort_keys(key, stream, n))
