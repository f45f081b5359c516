"""O4-O7 -- pool geometry, block / page tables, shuffled views, re-layout, tensor order.

Paper: Tier 2 "randomizes the mapping of virtual addresses to physical HBM pages" at 2 MB
granularity through the CUDA VMM API so that "tensor pointers and access semantics remain
unchanged" (Table 1b); Tier 1 permutes "the order in which tensors are
transferred and mapped" (Table 1a).  BJ:north_star (a) refines Tier 2 to
"a page/block-granular shuffle that scatters each layer's weight bytes into a randomly ordered
pool of physical pages".  Everything concrete below is reading O4-O7 / G3-G5 of SURVEY.md.

All byte buffers are 1-D numpy uint8 arrays.
"""
from dataclasses import dataclass
import numpy as np
from .keygen import keygen, STREAM_BLOCK, STREAM_PAGE, STREAM_TENSOR


@dataclass(frozen=True)
class PoolGeometry:
    B: int        # payload bytes
    b: int        # block bytes
    P: int        # page bytes
    nb: int       # ceil(B / b)      logical blocks
    bpp: int      # P / b            blocks per page
    npages: int   # ceil(nb / bpp)
    nslots: int   # npages * bpp     physical block slots


def pool_geometry(B, b, P):
    """O4: require b % 16 == 0 and P % b == 0."""
    if B < 1 or b < 16 or b % 16 or P % b:
        raise ValueError("bad pool geometry")
    nb = -(-B // b)
    bpp = P // b
    npages = -(-nb // bpp)
    return PoolGeometry(B, b, P, nb, bpp, npages, npages * bpp)


@dataclass(frozen=True)
class PoolTables:
    blockperm: np.ndarray
    blockinv: np.ndarray
    pageperm: np.ndarray
    pageinv: np.ndarray
    T_vmm: np.ndarray        # T[i] = blockinv[i], i < nb        (kernels address the VA view V)
    T_emulated: np.ndarray   # T[i] addresses the dump view D    (pool memory *is* D)


def pool_tables(key, g, identity=False):
    """O4 tables + O5 authorised tables.  identity=True: the "native" layout (all identity)."""
    if identity:
        ib = np.arange(g.nslots, dtype=np.uint32)
        ip = np.arange(g.npages, dtype=np.uint32)
        blockperm, blockinv, pageperm, pageinv = ib, ib.copy(), ip, ip.copy()
    else:
        blockperm, blockinv = keygen(key, STREAM_BLOCK, g.nslots)
        pageperm, pageinv = keygen(key, STREAM_PAGE, g.npages)
    s = blockinv[:g.nb].astype(np.int64)
    T_vmm = s.astype(np.uint32)
    T_emu = (pageinv[s // g.bpp].astype(np.int64) * g.bpp + s % g.bpp).astype(np.uint32)
    return PoolTables(blockperm, blockinv, pageperm, pageinv, T_vmm, T_emu)


def _padded_blocks(data, b):
    """data (uint8) zero-extended to a whole number of blocks, shaped [blocks, b]."""
    data = np.asarray(data, dtype=np.uint8).ravel()
    nblk = -(-data.size // b)
    out = np.zeros(nblk * b, dtype=np.uint8)
    out[:data.size] = data
    return out.reshape(nblk, b)


def shuffle_va(L, g, blockinv):
    """O5 VA view: V[blockinv[i]*b + o] = L[i*b + o] for i < nb; every other slot all zero."""
    Lb = _padded_blocks(L, g.b)
    assert Lb.shape[0] == g.nb
    V = np.zeros((g.nslots, g.b), dtype=np.uint8)
    for i in range(g.nb):
        V[int(blockinv[i])] = Lb[i]
    return V.ravel()


def dump_view(V, g, pageinv):
    """O5 dump view: D[pageinv[v]*P + o] = V[v*P + o] (what reading pages in physical order sees)."""
    Vp = np.asarray(V, dtype=np.uint8).reshape(g.npages, g.P)
    D = np.zeros_like(Vp)
    for v in range(g.npages):
        D[int(pageinv[v])] = Vp[v]
    return D.ravel()


def shuffle_into(pool, T, data, logical_offset, b):
    """cloak_shuffle on a sub-range: arena bytes [logical_offset, +len(data)) <- data.

    logical_offset is a block multiple; the last block is zero-padded (G4).  pool is modified in
    place; T is the authorised table of that pool (T_vmm for V, T_emulated for D).
    """
    if logical_offset % b:
        raise ValueError("logical_offset must be a block multiple")
    blocks = _padded_blocks(data, b)
    pv = pool.reshape(-1, b)
    first = logical_offset // b
    for j in range(blocks.shape[0]):
        pv[int(T[first + j])] = blocks[j]
    return pool


def unshuffle(pool, T, B, b, logical_offset=0, nbytes=None):
    """O5: L'[i*b + o] = pool[T[i]*b + o], truncated to the requested range."""
    if nbytes is None:
        nbytes = B - logical_offset
    if logical_offset % b:
        raise ValueError("logical_offset must be a block multiple")
    pv = np.asarray(pool, dtype=np.uint8).reshape(-1, b)
    first = logical_offset // b
    nblk = -(-nbytes // b)
    out = np.empty((nblk, b), dtype=np.uint8)
    for j in range(nblk):
        out[j] = pv[int(T[first + j])]
    return out.ravel()[:nbytes].copy()


def relayout(pool_A, T_A, T_B, g):
    """O6: the pool under key B that equals shuffle_B(unshuffle_A(pool_A)), zero pad slots included.

    T_A / T_B are the authorised tables (same kind) of the two pools; same B, b, P.
    """
    L = unshuffle(pool_A, T_A, g.B, g.b)
    out = np.zeros(g.nslots * g.b, dtype=np.uint8)
    return shuffle_into(out, T_B, L, 0, g.b)


def rekey_pages(D, g, pageinv_old, pageinv_new):
    """NEXT-1: the physical page map re-drawn, the VA view untouched ("periodically randomizes the mapping of
    virtual addresses to physical HBM pages"; "tensor pointers and access semantics remain unchanged").

    D is the dump view under the old page map.  VA page v sat on physical page pageinv_old[v] and sits on
    pageinv_new[v] afterwards:   D'[pageinv_new[v]*P + o] = D[pageinv_old[v]*P + o]   for every VA page v.
    """
    D = np.asarray(D, dtype=np.uint8)
    out = np.empty_like(D)
    for v in range(g.npages):
        src, dst = int(pageinv_old[v]) * g.P, int(pageinv_new[v]) * g.P
        out[dst:dst + g.P] = D[src:src + g.P]
    return out


def arena_plan(key, sizes, b):
    """O7 tensor order: offsets[t] for tensors of sizes[t] bytes, each padded to a block multiple.

    (order, _) = keygen(key, TENSOR, T); the arena holds order[0], order[1], ... back to back.
    Returns (offsets, total, order).
    """
    T = len(sizes)
    order, _ = keygen(key, STREAM_TENSOR, T)
    offsets = [0] * T
    at = 0
    for p in range(T):
        t = int(order[p])
        offsets[t] = at
        at += -(-int(sizes[t]) // b) * b
    return offsets, at, order


def adjacent_fraction(T):
    """G8 (reported only): fraction of logical neighbours (i, i+1) still adjacent: T[i+1] == T[i]+1."""
    T = np.asarray(T, dtype=np.int64)
    if T.size < 2:
        return 0.0
    return float(np.count_nonzero(T[1:] - T[:-1] == 1)) / (T.size - 1)


def run_lengths(T):
    """NEXT-3: lengths of the maximal runs i, i+1, ... of logically consecutive items with T[i+1] == T[i] + 1, in order.
    (the paper's contiguity metric counts address ranges that stayed physically contiguous.)"""
    T = [int(x) for x in np.asarray(T).ravel()]
    out, cur = [], 0
    for i in range(len(T)):
        if i > 0 and T[i] == T[i - 1] + 1:
            cur += 1
        else:
            if cur:
                out.append(cur)
            cur = 1
    if cur:
        out.append(cur)
    return out


def run_stats(T):
    """What cloak_pool_layout_report returns for one sequence: items, runs, longest run, items in runs of >= 2, the
    adjacent-pair fraction, and the histogram by power of two (bucket k: 2^k <= L < 2^(k+1))."""
    L = run_lengths(T)
    n = sum(L)
    hist = {}
    for x in L:
        k = x.bit_length() - 1
        hist[k] = hist.get(k, 0) + 1
    return dict(items=n, runs=len(L), longest_run=max(L) if L else 0, items_in_runs_of_2_or_more=sum(x for x in L if x >= 2),
                adjacent_fraction=(n - len(L)) / (n - 1) if n > 1 else 0.0, histogram=hist)
