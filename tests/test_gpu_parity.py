"""GPU parity: the CUDA library (through the C ABI binding) against the CPU oracle, element by element.

Integer / byte / index work must be bit-exact.  GEMV / GEMM outputs: O12 norm-wise error <= 2e-2 (bf16) and
<= 1e-5 (fp32), the tolerances BASELINE.json's north_star states, AND the element-wise bound that follows from the
arithmetic (util.check_linear), so that a dropped k-step cannot hide under 2e-2.  Both O12 errors of
every case are printed in the session summary (conftest.py) and written to gpurun_out/parity_errors.txt.
"""
import numpy as np
import pytest
import torch

import oracle as O
from synth import gen
from util import check_linear

pytestmark = pytest.mark.gpu

if torch.cuda.is_available():
    import paper_2606_18400_b200 as C
    from synth import cuda as synth_cuda
    from gpu_util import (Pool, dev_bytes, to_dev_bytes, to_host_bytes, bf16_dev_from_bits, bits_from_bf16_dev)

TOL = {"bf16": 2e-2, "f32": 1e-5}


# ------------------------------------------------------------------ harness twin
@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_synth_twins_agree(dtype):
    n, start = 100003, (1 << 32) + 12345
    t = torch.empty(n, dtype=torch.float32 if dtype == "f32" else torch.bfloat16, device="cuda")
    for kind in (gen.KIND_WEIGHT, gen.KIND_NORMAL):
        synth_cuda.fill(t, 7, 3, kind=kind, start=start)
        ref = gen.synth(7, 3, (n,), dtype, kind=kind, start=start)
        got = t.cpu().numpy() if dtype == "f32" else bits_from_bf16_dev(t)
        assert np.array_equal(got, ref)


# ------------------------------------------------------------------ S1 keygen
@pytest.mark.parametrize("n", [1, 2, 8, 16, 256, 1024, 4096, 4097, 14336, 245056, 1 << 20, (1 << 20) + 77,
                               (1 << 24) + 3])      # the last one: more elements than 4 x the 2^22 bucket cap
def test_keygen_bit_exact(n):
    perm = torch.empty(n, dtype=torch.int32, device="cuda")
    inv = torch.empty(n, dtype=torch.int32, device="cuda")
    for key, stream in [(0x1234, 0), (0xDEADBEEF12345678, (5 << 32) | 9)]:
        C.cloak_keygen(key, stream, n, perm, inv)
        rp, ri = O.keygen(key, stream, n)
        assert np.array_equal(perm.cpu().numpy().view(np.uint32), rp)
        assert np.array_equal(inv.cpu().numpy().view(np.uint32), ri)
    C.cloak_keygen(0x1234, 0, n, perm, None)          # either output may be NULL
    inv.zero_()
    C.cloak_keygen(0x1234, 0, n, None, inv)
    rp, ri = O.keygen(0x1234, 0, n)
    assert np.array_equal(perm.cpu().numpy().view(np.uint32), rp)
    assert np.array_equal(inv.cpu().numpy().view(np.uint32), ri)


# ------------------------------------------------------------------ S2/S4 pool, shuffle, unshuffle
POOLS = [
    # (payload, block, page, flags)             what it covers
    (1 << 20, 4096, 65536, 0),                   # cfg0 one matrix: 256 blocks, 16 emulated 64 KiB pages
    (3 << 20, 4096, 65536, 0),                   # cfg0 three matrices: 768 blocks, 48 pages
    ((1 << 20) + 4096 * 3 + 1040, 4096, 65536, 0),   # ragged: partial last block, partial last page
    (5 << 20, 65536, 2 << 20, 0),                # real VMM pages, partial last page
    (7 * 65536 + 512, 65536, 2 << 20, 0),        # real VMM, single page, ragged
    (6 << 20, 1 << 20, 2 << 20, 2),              # PLAIN_ALLOC with 2 MiB pages (emulated)
    (4 << 20, 2 << 20, 2 << 20, 0),              # block == page
    (100 * 256, 256, 1024, 0),                   # tiny blocks (LDG engine only)
]


@pytest.mark.parametrize("engine", [1, 2])
@pytest.mark.parametrize("payload,block,page,flags", POOLS)
def test_shuffle_unshuffle_bit_exact(payload, block, page, flags, engine):
    key = 0x1234
    g = O.pool_geometry(payload, block, page)
    t = O.pool_tables(key, g)
    L = np.random.default_rng(payload).integers(0, 256, payload, dtype=np.uint8)
    C.cloak_set_copy_engine(engine)
    try:
        with Pool(payload, block, page, key, flags) as p:
            assert (p.info["nb"], p.info["nslots"], p.info["npages"]) == (g.nb, g.nslots, g.npages)
            bp, bi, pp, pi = p.tables()
            assert np.array_equal(bp, t.blockperm) and np.array_equal(bi, t.blockinv)
            assert np.array_equal(pp, t.pageperm) and np.array_equal(pi, t.pageinv)
            vmm = p.info["is_vmm"]
            assert vmm == (page % (2 << 20) == 0 and not (flags & 2))
            assert np.array_equal(p.table_T(), t.T_vmm if vmm else t.T_emulated)
            dL = to_dev_bytes(L)
            padded = (payload + 15) // 16 * 16
            if padded != payload:
                dL = torch.cat([dL, dev_bytes(padded - payload)])
            C.cloak_shuffle(p.h, dL, 0, padded)
            V = O.shuffle_va(L, g, t.blockinv)
            D = O.dump_view(V, g, t.pageinv)
            assert np.array_equal(p.raw(), V if vmm else D)       # zero pad slots are compared too (G4)
            assert np.array_equal(p.dump(), D)                    # physical-order view (alias mapping for VMM)
            out = dev_bytes(padded)
            C.cloak_unshuffle(p.h, out, 0, padded)
            assert np.array_equal(out.cpu().numpy()[:payload], L)
            # a sub-range: blocks [1, 3) plus a 48-byte tail of the next
            if g.nb >= 4:
                sub = dev_bytes(2 * block + 48)
                C.cloak_unshuffle(p.h, sub, block, 2 * block + 48)
                assert np.array_equal(sub.cpu().numpy(), L[block:3 * block + 48])
    finally:
        C.cloak_set_copy_engine(0)


def test_shuffle_by_tensor_ranges_and_zero_padding():
    """Tensors placed by cloak_arena_plan, each shuffled on its own; padding after a short tensor is zero."""
    block, page, key = 4096, 65536, 0x1234
    sizes = [5000 * 16, 4096 * 3, 16, 70000 * 16 // 16 * 16]
    offs, total = C.cloak_arena_plan(key, sizes, block)
    o_offs, o_total, _ = O.arena_plan(key, sizes, block)
    assert offs == o_offs and total == o_total
    g = O.pool_geometry(total, block, page)
    t = O.pool_tables(key, g)
    rng = np.random.default_rng(0)
    datas = [rng.integers(1, 256, s, dtype=np.uint8) for s in sizes]
    ref = np.zeros(g.nslots * block, np.uint8)
    with Pool(total, block, page, key) as p:
        for d, o in zip(datas, offs):
            C.cloak_shuffle(p.h, to_dev_bytes(d), o, d.size)
            O.shuffle_into(ref, t.T_emulated, d, o, block)
        assert np.array_equal(p.raw(), ref)


@pytest.mark.parametrize("payload,block,page", [(3 << 20, 4096, 65536), (40 << 20, 65536, 2 << 20), (1 << 20, 256, 1024)])
def test_pool_adjacency_matches_the_oracle(payload, block, page):
    """NEXT-3 layout-quality report: adjacent-block / adjacent-page fractions equal oracle.adjacent_fraction."""
    g = O.pool_geometry(payload, block, page)
    t = O.pool_tables(0x1234, g)
    with Pool(payload, block, page, 0x1234) as p, Pool(payload, block, page, 0x1234, C.CLOAK_POOL_IDENTITY) as pi:
        a = C.cloak_pool_adjacency(p.h)
        assert a["va_blocks"] == pytest.approx(O.adjacent_fraction(t.T_vmm), abs=1e-15)
        assert a["physical_blocks"] == pytest.approx(O.adjacent_fraction(t.T_emulated), abs=1e-15)
        assert a["pages"] == pytest.approx(O.adjacent_fraction(t.pageinv), abs=1e-15)
        assert a["physical_blocks"] < 0.02                          # G8: about 1 / nslots for a uniform permutation
        assert C.cloak_pool_adjacency(pi.h) == dict(va_blocks=1.0, physical_blocks=1.0, pages=1.0)


@pytest.mark.parametrize("payload,block,page,flags", [(3 << 20, 4096, 65536, 0), (300 << 20, 65536, 2 << 20, 0), (1 << 20, 256, 1024, 0),
                                                      ((37 << 20) + 4096, 4096, 2 << 20, 0), (40 << 20, 65536, 2 << 20, 1)])
def test_pool_layout_report_matches_the_oracle(payload, block, page, flags):
    """NEXT-3: runs of logically consecutive blocks / pages that stayed consecutive (VA view, physical view, page map) --
    counts, longest run, histogram by power of two -- against oracle.run_stats on the oracle's own tables; an identity pool
    (flags = 1) is one run of everything.  After a page re-key the report follows the new page map."""
    key = 0x1234
    g = O.pool_geometry(payload, block, page)
    t = O.pool_tables(key, g)

    def check(rep, blockinv, pageinv):
        phys = [int(pageinv[int(s) // g.bpp]) * g.bpp + int(s) % g.bpp for s in blockinv[:g.nb]]
        for name, seq in (("va_blocks", blockinv[:g.nb]), ("physical_blocks", phys), ("pages", pageinv)):
            ref = O.run_stats(seq)
            got = rep[name]
            assert {k: got[k] for k in ("items", "runs", "longest_run", "items_in_runs_of_2_or_more")} == \
                   {k: ref[k] for k in ("items", "runs", "longest_run", "items_in_runs_of_2_or_more")}, name
            assert abs(got["adjacent_fraction"] - ref["adjacent_fraction"]) < 1e-12
            assert got["histogram"] == {f"2^{k}": c for k, c in ref["histogram"].items()}, name
    with Pool(payload, block, page, key, flags) as p:
        rep = C.cloak_pool_layout_report(p.h)
        if flags & C.CLOAK_POOL_IDENTITY:
            check(rep, np.arange(g.nslots), np.arange(g.npages))
            assert rep["physical_blocks"]["runs"] == 1 and rep["pages"]["longest_run"] == g.npages
        else:
            check(rep, t.blockinv, t.pageinv)
            adj = C.cloak_pool_adjacency(p.h)
            assert abs(adj["physical_blocks"] - rep["physical_blocks"]["adjacent_fraction"]) < 1e-12
            if p.info["is_vmm"]:
                C.cloak_rekey_pages_begin(p.h, 0x5678, 2)
                C.cloak_rekey_pages_finish(p.h)
                check(C.cloak_pool_layout_report(p.h), t.blockinv, O.pool_tables(0x5678, g).pageinv)


@pytest.mark.parametrize("block,page,n", [(4096, 65536, 5), (65536, 2 << 20, 150), (256, 1024, 4)])
def test_shuffle_many_equals_one_call_per_range(block, page, n):
    """cloak_shuffle_many / cloak_unshuffle_many: n tensors of mixed sizes (ragged tails, > 128 ranges -> two launches) in
    one call leave the pool exactly as the oracle's shuffle_into of each, and come back bit for bit."""
    key = 0x1234
    rng = np.random.default_rng(5)
    sizes = [int(rng.integers(1, 40)) * block // 2 // 16 * 16 + (16 if i % 3 == 0 else 0) for i in range(n)]
    offs, total = C.cloak_arena_plan(key, sizes, block)
    g = O.pool_geometry(total, block, page)
    t = O.pool_tables(key, g)
    datas = [rng.integers(1, 256, s_, dtype=np.uint8) for s_ in sizes]
    with Pool(total, block, page, key) as p:
        T = t.T_vmm if p.info["is_vmm"] else t.T_emulated
        ref = np.zeros(g.nslots * block, np.uint8)
        for d, o in zip(datas, offs):
            O.shuffle_into(ref, T, d, o, block)
        dev = [to_dev_bytes(d) for d in datas]
        C.cloak_shuffle_many(p.h, dev, offs, sizes)
        assert np.array_equal(p.raw(), ref)
        outs = [dev_bytes(s_) for s_ in sizes]
        C.cloak_unshuffle_many(p.h, outs, offs, sizes)
        for d, o_ in zip(datas, outs):
            assert np.array_equal(o_.cpu().numpy(), d)
        with pytest.raises(C.CloakError):
            C.cloak_shuffle_many(p.h, dev[:1], [offs[0] + 16], sizes[:1])        # offset not a block multiple


def test_identity_pool_is_the_native_layout():
    payload, block, page = 3 << 20, 65536, 2 << 20
    L = np.random.default_rng(3).integers(0, 256, payload, dtype=np.uint8)
    for flags in (C.CLOAK_POOL_IDENTITY, C.CLOAK_POOL_IDENTITY | C.CLOAK_POOL_PLAIN_ALLOC):
        with Pool(payload, block, page, 0x1234, flags) as p:
            C.cloak_shuffle(p.h, to_dev_bytes(L), 0, payload)
            raw = p.raw()
            assert np.array_equal(raw[:payload], L) and not raw[payload:].any()
            assert np.array_equal(p.table_T(), np.arange(p.info["nb"], dtype=np.uint32))


@pytest.mark.parametrize("engine", [1, 2])
@pytest.mark.parametrize("payload,block,page", [(3 << 20, 4096, 65536), (5 << 20, 65536, 2 << 20),
                                                ((2 << 20) + 4096 * 5 + 160, 4096, 2 << 20)])
def test_relayout_bit_exact(payload, block, page, engine):
    ka, kb = 0x1234, 0x5678
    g = O.pool_geometry(payload, block, page)
    ta, tb = O.pool_tables(ka, g), O.pool_tables(kb, g)
    L = np.random.default_rng(11).integers(0, 256, payload, dtype=np.uint8)
    padded = (payload + 15) // 16 * 16
    C.cloak_set_copy_engine(engine)
    try:
        with Pool(payload, block, page, ka) as pa, Pool(payload, block, page, kb) as pb:
            vmm = pa.info["is_vmm"]
            TA, TB = (ta.T_vmm, tb.T_vmm) if vmm else (ta.T_emulated, tb.T_emulated)
            dL = torch.cat([to_dev_bytes(L), dev_bytes(padded - payload)]) if padded != payload else to_dev_bytes(L)
            C.cloak_shuffle(pa.h, dL, 0, padded)
            ref_a = pa.raw()
            C.cloak_relayout(pa.h, pb.h)
            assert np.array_equal(pb.raw(), O.relayout(ref_a, TA, TB, g))       # = shuffle_B(unshuffle_A)
            with Pool(payload, block, page, ka) as pa2:
                C.cloak_relayout(pb.h, pa2.h)                                   # A -> B -> A restores pool A
                assert np.array_equal(pa2.raw(), ref_a)
    finally:
        C.cloak_set_copy_engine(0)


@pytest.mark.parametrize("payload,block,page,spare", [
    (3 << 20, 4096, 65536, 0),                     # emulated pages, one page of spare
    ((1 << 20) + 4096 * 3 + 1040, 4096, 65536, 4096),   # ragged payload, a single spare block: one long chain per cycle
    (40 << 20, 65536, 2 << 20, 0),                 # real VMM pages
    (40 << 20, 65536, 2 << 20, 16 << 20),          # lots of spare: many short segments
    (100 * 256, 256, 1024, 0),                     # tiny blocks
])
def test_rekey_inplace_equals_oracle_relayout(payload, block, page, spare):
    """NEXT-1: cloak_rekey_inplace leaves the pool exactly as the oracle's relayout(pool, T_A, T_B) over the unchanged page
    map, the tables are key B's block tables + key A's page tables, and reads through the new table give the data."""
    key_a, key_b = 0x1234, 0x5678
    g = O.pool_geometry(payload, block, page)
    ta, tb = O.pool_tables(key_a, g), O.pool_tables(key_b, g)
    L = np.random.default_rng(11).integers(0, 256, payload, dtype=np.uint8)
    padded = (payload + 15) // 16 * 16
    dL = torch.cat([to_dev_bytes(L), dev_bytes(padded - payload)]) if padded != payload else to_dev_bytes(L)
    with Pool(payload, block, page, key_a) as p:
        vmm = p.info["is_vmm"]
        C.cloak_shuffle(p.h, dL, 0, padded)
        before = p.raw()
        # O5 over an unchanged page map: the memory slot of logical block i under key B
        sb = tb.blockinv[:g.nb].astype(np.int64)
        T_b = tb.T_vmm if vmm else (ta.pageinv[sb // g.bpp].astype(np.int64) * g.bpp + sb % g.bpp).astype(np.uint32)
        T_a = ta.T_vmm if vmm else ta.T_emulated
        C.cloak_rekey_inplace(p.h, key_b, spare)
        assert np.array_equal(p.raw(), O.relayout(before, T_a, T_b, g))
        bp, bi, pp, pinv = p.tables()
        assert np.array_equal(bp, tb.blockperm) and np.array_equal(bi, tb.blockinv)
        assert np.array_equal(pp, ta.pageperm) and np.array_equal(pinv, ta.pageinv)
        assert np.array_equal(p.table_T(), T_b)
        out = dev_bytes(padded)
        C.cloak_unshuffle(p.h, out, 0, padded)
        assert np.array_equal(out.cpu().numpy()[:payload], L)
        C.cloak_rekey_inplace(p.h, key_b, spare)                   # same key again: nothing moves
        assert np.array_equal(p.table_T(), T_b)
        C.cloak_rekey_inplace(p.h, key_a, spare)                   # and back
        assert np.array_equal(p.raw(), before)


@pytest.mark.parametrize("payload,block,page,spares,per_step", [
    (40 << 20, 65536, 2 << 20, 1, 1),        # 20 pages, one spare page, one move per step: the minimal-memory form
    (300 << 20, 65536, 2 << 20, 4, 4),       # 150 pages, 4 cycles in flight
    (37 << 20, 4096, 2 << 20, 3, 16),        # ragged payload (zero pad slots move with their pages), small blocks
])
def test_rekey_pages_under_live_gemv(payload, block, page, spares, per_step):
    """NEXT-1: cloak_rekey_pages_begin / _step between GEMV launches (plain and CUDA-graph replays captured BEFORE the
    re-key).  During and after: every GEMV output bit-identical to the one before the re-key, the logical bytes unchanged;
    after: page tables == the oracle's keygen(new_key, PAGE), dump view == oracle.rekey_pages(D before), V unchanged as read
    through cloak_unshuffle; a second re-key (pages travel back through the first half) and _finish (stop-the-world) too."""
    key, seed = 0x1234, 9
    g = O.pool_geometry(payload, block, page)
    N, K = 512, 1024
    Wm = gen.synth(seed, 0, (N, K), "bf16")
    X = gen.synth(seed + 100, 0, (4, K), "bf16", kind=gen.KIND_NORMAL)
    rng = np.random.default_rng(seed)
    L = rng.integers(0, 256, payload, dtype=np.uint8)
    w_off = (payload // 2) // block * block
    L[w_off:w_off + N * K * 2] = Wm.view(np.uint8).ravel()                   # a weight matrix in the middle of the arena
    with Pool(payload, block, page, key) as p:
        assert p.info["is_vmm"]
        dL = to_dev_bytes(L)
        C.cloak_shuffle(p.h, dL, 0, payload)
        t_old = O.pool_tables(key, g)
        D0 = p.dump()
        assert np.array_equal(D0, O.dump_view(O.shuffle_va(L, g, t_old.blockinv), g, t_old.pageinv))
        dX = bf16_dev_from_bits(X)
        w = C.cloak_tensor(w_off, N, K, C.CLOAK_BF16, C.CLOAK_ROWMAJOR)
        y0 = torch.zeros(4, N, dtype=torch.bfloat16, device="cuda")
        C.cloak_gemv(p.h, w, dX, y0, 4)
        check_linear(y0.float().cpu().numpy(), X, Wm, "bf16", f"rekey_pages:{g.npages}pages:before", TOL["bf16"])
        yg = torch.zeros_like(y0)
        gph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(gph):
            C.cloak_gemv(p.h, w, dX, yg, 4)
        D_prev, inv_prev = D0, t_old.pageinv
        for new_key, use_finish in ((0x5678, False), (0x9abc, False), (0x1234, True)):
            C.cloak_rekey_pages_begin(p.h, new_key, spares)
            steps = 0
            while True:
                if use_finish:
                    C.cloak_rekey_pages_finish(p.h)                           # the stop-the-world form
                    left = C.cloak_rekey_pages_step(p.h, 1)
                    assert left == 0
                else:
                    left = C.cloak_rekey_pages_step(p.h, per_step)           # non-blocking, between GEMV launches
                y = torch.zeros_like(y0)
                C.cloak_gemv(p.h, w, dX, y, 4)                                # reads through the table as it stands now
                yg.zero_()
                gph.replay()                                                  # captured before any page moved
                if steps % 7 == 0 or not left:
                    torch.cuda.synchronize()
                    assert torch.equal(y, y0) and torch.equal(yg, y0), (hex(new_key), steps)
                steps += 1
                if not left:
                    break
                assert steps < 50 * g.npages, "the page re-key does not terminate"
            torch.cuda.synchronize()
            t_new = O.pool_tables(new_key, g)
            _, _, pp, pinv = p.tables()
            assert np.array_equal(pp, t_new.pageperm) and np.array_equal(pinv, t_new.pageinv)
            D1 = p.dump()
            assert np.array_equal(D1, O.rekey_pages(D_prev, g, inv_prev, t_new.pageinv)), hex(new_key)
            back = dev_bytes(payload)
            C.cloak_unshuffle(p.h, back, 0, payload)
            assert np.array_equal(to_host_bytes(back), L)                     # the logical view never changed
            D_prev, inv_prev = D1, t_new.pageinv
        # the block re-key still works on a pool whose pages sit in either half, and then a fresh shuffle
        C.cloak_rekey_inplace(p.h, 0x7777, 0)
        back = dev_bytes(payload)
        C.cloak_unshuffle(p.h, back, 0, payload)
        assert np.array_equal(to_host_bytes(back), L)
        y = torch.zeros_like(y0)
        C.cloak_gemv(p.h, w, dX, y, 4)
        torch.cuda.synchronize()
        assert torch.equal(y, y0)
        del gph


@pytest.mark.parametrize("payload,block,page", [(16, 16, 16), (48, 16, 64), (100 * 16, 16, 16), (2 << 20, 2 << 20, 2 << 20), (4096, 65536, 2 << 20),
                                                (1 << 20, 65536, 2 << 20)])
def test_degenerate_pools(payload, block, page):
    """The smallest and the most lopsided pools: one slot (b = P = B: a plain copy), a payload shorter than a block and a page,
    pages of one block, one real 2 MiB page holding one 2 MiB block, a real page mostly padding.  Tables, V, D, the round
    trip, the layout report and (real pages) a page re-key that has nothing or almost nothing to move."""
    key = 0x1234
    g = O.pool_geometry(payload, block, page)
    t = O.pool_tables(key, g)
    L = np.random.default_rng(payload).integers(0, 256, payload, dtype=np.uint8)
    with Pool(payload, block, page, key) as p:
        bp, bi, pp, pinv = p.tables()
        assert np.array_equal(bp, t.blockperm) and np.array_equal(pinv, t.pageinv)
        dL = to_dev_bytes(L)
        C.cloak_shuffle(p.h, dL, 0, payload)
        V = O.shuffle_va(L, g, t.blockinv)
        D = O.dump_view(V, g, t.pageinv)
        assert np.array_equal(p.dump(), D)
        assert np.array_equal(p.raw(), V if p.info["is_vmm"] else D)
        back = dev_bytes(payload)
        C.cloak_unshuffle(p.h, back, 0, payload)
        assert np.array_equal(to_host_bytes(back), L)
        rep = C.cloak_pool_layout_report(p.h)
        assert rep["pages"]["items"] == g.npages and rep["va_blocks"]["items"] == g.nb
        assert rep["va_blocks"]["runs"] == O.run_stats(t.blockinv[:g.nb])["runs"]
        if p.info["is_vmm"]:
            C.cloak_rekey_pages_begin(p.h, 0x5678, 1)
            C.cloak_rekey_pages_finish(p.h)
            t2 = O.pool_tables(0x5678, g)
            assert np.array_equal(p.tables()[3], t2.pageinv)
            assert np.array_equal(p.dump(), O.rekey_pages(D, g, t.pageinv, t2.pageinv))
            back.zero_()
            C.cloak_unshuffle(p.h, back, 0, payload)
            assert np.array_equal(to_host_bytes(back), L)


def test_host_buffer_round_trip():
    payload, block, page, key = (5 << 20) + 4096 + 32, 4096, 2 << 20, 0x1234
    g = O.pool_geometry(payload, block, page)
    t = O.pool_tables(key, g)
    L = np.random.default_rng(21).integers(0, 256, payload, dtype=np.uint8)
    hL = torch.from_numpy(L.copy()).pin_memory()
    out = torch.zeros(payload, dtype=torch.uint8).pin_memory()
    with Pool(payload, block, page, key) as p:
        C.cloak_shuffle_host(p.h, hL, 0, payload)
        assert np.array_equal(p.raw(), O.shuffle_va(L, g, t.blockinv))
        C.cloak_unshuffle_host(p.h, out, 0, payload)
        assert np.array_equal(out.numpy(), L)


# ------------------------------------------------------------------ S5 neuron / head permutation
def _dev(a, dtype):
    return torch.from_numpy(a.copy()).cuda() if dtype == "f32" else bf16_dev_from_bits(a)


def _host(t, dtype):
    return t.cpu().numpy() if dtype == "f32" else bits_from_bf16_dev(t)


PERM_SHAPES = [
    # hidden, inter, n_q, n_kv, d, dtype, layer
    (256, 1024, 4, 4, 64, "f32", 0),        # cfg0's MLP block (+ an MHA head set, G = 1)
    (256, 1000, 8, 2, 32, "bf16", 3),       # ragged inter, GQA
    (4096, 14336, 32, 8, 128, "bf16", 0),   # cfg1 at full size
    (640, 1536, 40, 8, 16, "bf16", 63),     # cfg3's head structure (40 q / 8 kv), non-power-of-two rows
]


@pytest.mark.parametrize("hidden,inter,n_q,n_kv,d,dtype,layer", PERM_SHAPES)
def test_permute_mlp_heads_bit_exact(hidden, inter, n_q, n_kv, d, dtype, layer):
    key, seed = 0x1234, 5
    shapes = dict(gate=(inter, hidden), up=(inter, hidden), down=(hidden, inter), q=(n_q * d, hidden),
                  k=(n_kv * d, hidden), v=(n_kv * d, hidden), o=(hidden, n_q * d))
    W = {nm: gen.synth(seed, i, shp, dtype) for i, (nm, shp) in enumerate(shapes.items())}
    dW = {nm: _dev(a, dtype) for nm, a in W.items()}
    dO = {nm: torch.zeros_like(t) for nm, t in dW.items()}
    sh = C.cloak_block_shape(hidden, inter, n_q, n_kv, d, C.CLOAK_F32 if dtype == "f32" else C.CLOAK_BF16, layer)
    C.cloak_permute_mlp_heads(key, sh, **dW, **{k + "_o": v for k, v in dO.items()})
    pi = O.mlp_perm(key, layer, inter)
    kappa, eta = O.head_maps(key, layer, n_q, n_kv)
    g2, u2, d2 = O.permute_mlp(W["gate"], W["up"], W["down"], pi)
    q2, k2, v2, o2 = O.permute_heads(W["q"], W["k"], W["v"], W["o"], kappa, eta, d)
    for nm, ref in dict(gate=g2, up=u2, down=d2, q=q2, k=k2, v=v2, o=o2).items():
        assert np.array_equal(_host(dO[nm], dtype), ref), nm
    # subsets: MLP only / heads only leave the other outputs untouched
    z = {nm: torch.zeros_like(t) for nm, t in dW.items()}
    C.cloak_permute_mlp_heads(key, sh, gate=dW["gate"], gate_o=z["gate"], o=dW["o"], o_o=z["o"])
    assert np.array_equal(_host(z["gate"], dtype), g2) and np.array_equal(_host(z["o"], dtype), o2)
    assert not z["down"].any() and not z["q"].any()


@pytest.mark.parametrize("hidden,inter,n_q,n_kv,d,dtype,layer,block,page", [
    (256, 1024, 4, 4, 64, "f32", 0, 4096, 65536),            # cfg0's block, emulated pages
    (256, 1000, 8, 2, 32, "bf16", 3, 4096, 65536),           # ragged inter: rows straddle blocks, partial last blocks
    (4096, 14336, 32, 8, 128, "bf16", 0, 65536, 2 << 20),    # cfg1 at full size, real VMM pages
    (640, 1536, 40, 8, 16, "bf16", 63, 1024, 65536),         # blocks smaller than a row
])
def test_fused_load_equals_permute_then_shuffle(hidden, inter, n_q, n_kv, d, dtype, layer, block, page):
    """cloak_load_mlp_heads: the pool bytes are the oracle's shuffle(permute(W)) -- and the two-pass GPU path's."""
    key, seed = 0x1234, 7
    e = 4 if dtype == "f32" else 2
    shapes = gen.layer_shapes(hidden, inter, n_q, n_kv, d)
    W = {nm: gen.synth(seed, i, shp, dtype) for i, (nm, shp) in enumerate(shapes)}
    dW = {nm: _dev(a, dtype) for nm, a in W.items()}
    sizes = [e * n * k for _, (n, k) in shapes]
    offs, total = C.cloak_arena_plan(key, sizes, block)
    off = {nm: o for (nm, _), o in zip(shapes, offs)}
    pi = O.mlp_perm(key, layer, inter)
    kappa, eta = O.head_maps(key, layer, n_q, n_kv)
    ref = dict(zip(("gate", "up", "down"), O.permute_mlp(W["gate"], W["up"], W["down"], pi)))
    ref.update(zip(("q", "k", "v", "o"), O.permute_heads(W["q"], W["k"], W["v"], W["o"], kappa, eta, d)))
    g = O.pool_geometry(total, block, page)
    t = O.pool_tables(key, g)
    sh = C.cloak_block_shape(hidden, inter, n_q, n_kv, d, C.CLOAK_F32 if dtype == "f32" else C.CLOAK_BF16, layer)
    with Pool(total, block, page, key) as pf, Pool(total, block, page, key) as p2:
        T = t.T_vmm if pf.info["is_vmm"] else t.T_emulated
        refpool = np.zeros(g.nslots * block, np.uint8)
        for nm, _ in shapes:
            O.shuffle_into(refpool, T, ref[nm].view(np.uint8).ravel(), off[nm], block)
        # stale bytes everywhere first: the fused path must leave exactly the oracle's pool, zero tails included
        junk = torch.full((total,), 0xA5, dtype=torch.uint8, device="cuda")
        C.cloak_shuffle(pf.h, junk, 0, total)
        C.cloak_load_mlp_heads(key, sh, pf.h, off, **dW)
        got = pf.raw()
        for (nm, _), sz in zip(shapes, sizes):                      # every block a tensor owns, padding included
            first, nblk = off[nm] // block, (sz + block - 1) // block
            for i in range(first, first + nblk):
                s0 = int(T[i]) * block
                assert np.array_equal(got[s0:s0 + block], refpool[s0:s0 + block]), (nm, i - first)
        dP = {nm: torch.zeros_like(x) for nm, x in dW.items()}
        C.cloak_permute_mlp_heads(key, sh, **dW, **{k + "_o": v for k, v in dP.items()})
        for nm, _ in shapes:
            C.cloak_shuffle(p2.h, dP[nm], off[nm], dP[nm].numel() * e)
        assert np.array_equal(p2.raw(), refpool)
        # a subset of the tensors only
        C.cloak_shuffle(pf.h, junk, 0, total)
        C.cloak_load_mlp_heads(key, sh, pf.h, off, down=dW["down"], k=dW["k"])
        got = pf.raw()
        for nm in ("down", "k"):
            i = off[nm] // block
            s0 = int(T[i]) * block
            assert np.array_equal(got[s0:s0 + block], refpool[s0:s0 + block])
        i = off["gate"] // block
        assert (got[int(T[i]) * block:int(T[i]) * block + block] == 0xA5).all()      # untouched


@pytest.mark.parametrize("layout,where,dtype,block", [("rowmajor", "pinned", "bf16", 4096), ("tile128", "pinned", "bf16", 65536),
                                                      ("tile128", "device", "f32", 65536), ("rowmajor", "device", "bf16", 256)])
def test_load_tensors_one_pass_from_host_or_device(layout, where, dtype, block):
    """NEXT-2: cloak_load_tensors -- two decoder layers' 14 tensors and a plain matrix, read once from PINNED HOST memory (the
    kernels themselves reach across PCIe) or from device memory, permuted, laid out (ROWMAJOR / TILE128) and scattered through
    the block table in one pass, listed in model order and issued in arena (keyed tensor) order: the pool's bytes equal the
    oracle's shuffle_into(to_tile128(permute(W))) for every tensor, unused slots and block tails zero."""
    key, seed, page = 0x1234, 11, 2 << 20
    H, I, nq, nkv, d = 256, 768, 4, 2, 64
    e = 4 if dtype == "f32" else 2
    shapes = gen.layer_shapes(H, I, nq, nkv, d)
    names = [(l, nm, shp) for l in (0, 5) for nm, shp in shapes] + [(0, "plain", (384, 256))]
    W = {(l, nm): gen.synth(seed, i, shp, dtype) for i, (l, nm, shp) in enumerate(names)}
    sizes = [shp[0] * shp[1] * e for _, _, shp in names]
    offs, total = C.cloak_arena_plan(key, sizes, block)
    g = O.pool_geometry(total, block, page)
    t = O.pool_tables(key, g)
    ref = np.zeros(g.nslots * block, np.uint8)
    for l in (0, 5):
        pi = O.mlp_perm(key, l, I)
        kappa, eta = O.head_maps(key, l, nq, nkv)
        pm = dict(zip(("gate", "up", "down"), O.permute_mlp(W[l, "gate"], W[l, "up"], W[l, "down"], pi)))
        pm.update(zip(("q", "k", "v", "o"), O.permute_heads(W[l, "q"], W[l, "k"], W[l, "v"], W[l, "o"], kappa, eta, d)))
        for nm in pm:
            W[l, nm + "'"] = pm[nm]
    W[0, "plain'"] = W[0, "plain"]
    for (l, nm, shp), o in zip(names, offs):
        a = W[l, nm + "'"]
        a = O.to_tile128(a) if layout == "tile128" else a
        O.shuffle_into(ref, t.T_vmm, np.ascontiguousarray(a).view(np.uint8).ravel(), o, block)
    keep = []

    def put(a):
        h = torch.from_numpy(np.ascontiguousarray(a).view(np.uint8).reshape(-1).copy())
        h = h.pin_memory() if where == "pinned" else h.cuda()
        keep.append(h)
        return h
    items = [(put(W[l, nm]), o, l, nm if nm != "plain" else "plain") + ((shp[0], shp[1]) if nm == "plain" else ())
             for (l, nm, shp), o in zip(names, offs)]
    sh = C.cloak_block_shape(H, I, nq, nkv, d, C.CLOAK_F32 if dtype == "f32" else C.CLOAK_BF16, 0)
    with Pool(total, block, page, key) as p:
        C.cloak_load_tensors(key, sh, p.h, items[::-1], C.CLOAK_TILE128 if layout == "tile128" else C.CLOAK_ROWMAJOR)   # any listing order
        torch.cuda.synchronize()
        assert np.array_equal(p.raw(), ref)
        # argument checks: overlap, bad role, unaligned offset, a pageable host source (the kernels could not read it)
        pageable = np.zeros(I * H * e + 64, np.uint8)
        pageable = pageable[(-pageable.ctypes.data) % 64:]
        for bad, st in (([items[0], items[0]], C.CLOAK_ERR_INVALID), ([(items[0][0], offs[0], 0, 9)], C.CLOAK_ERR_INVALID),
                        ([(items[0][0], offs[0] + 16, 0, "gate")], C.CLOAK_ERR_ALIGN),
                        ([(pageable, offs[names.index((0, "gate", (I, H)))], 0, "gate")], C.CLOAK_ERR_INVALID)):
            with pytest.raises(C.CloakError) as ei:
                C.cloak_load_tensors(key, sh, p.h, bad)
            assert ei.value.status == st


def test_tile128_bit_exact():
    for dtype, (N, K) in [("bf16", (256, 384)), ("f32", (128, 256)), ("bf16", (1024, 5120))]:
        W = gen.synth(9, 0, (N, K), dtype)
        src = _dev(W, dtype)
        dst = torch.zeros_like(src).reshape(-1)
        C.cloak_to_tile128(src, dst, N, K, C.CLOAK_F32 if dtype == "f32" else C.CLOAK_BF16)
        assert np.array_equal(_host(dst, dtype), O.to_tile128(W))


# ------------------------------------------------------------------ S6 cloaked GEMV
def _load_pool(p, tensors, offs, dtype):
    for (nm, a), o in zip(tensors, offs):
        d = _dev(a, dtype)
        C.cloak_shuffle(p.h, d, o, d.numel() * d.element_size())


GEMV_CASES = [
    # dtype, block, page, shapes [(N, K)], batches
    ("f32", 4096, 65536, [(1024, 256), (1024, 256), (256, 1024)], [1, 3]),                 # cfg0
    ("bf16", 4096, 65536, [(64, 256), (256, 128), (48, 1024)], [1, 4, 8, 9, 16]),          # several tiles, ragged N/16
    ("bf16", 65536, 2 << 20, [(1024, 4096), (4096, 14336)], [1, 4, 16]),                   # cfg1's k and down shapes
    ("bf16", 65536, 2 << 20, [(5120, 5120), (1024, 5120)], [1, 16]),                       # cfg3's non-power-of-two rows
]


@pytest.mark.parametrize("dtype,block,page,shapes,batches", GEMV_CASES)
def test_gemv_vs_oracle_and_identity_bit_identical(dtype, block, page, shapes, batches):
    key, seed = 0x1234, 1
    e = 4 if dtype == "f32" else 2
    dt = C.CLOAK_F32 if dtype == "f32" else C.CLOAK_BF16
    tensors = [(f"t{i}", gen.synth(seed, i, shp, dtype)) for i, shp in enumerate(shapes)]
    sizes = [a.size * e for _, a in tensors]
    offs, total = C.cloak_arena_plan(key, sizes, block)
    with Pool(total, block, page, key) as pc, Pool(total, block, page, key, C.CLOAK_POOL_IDENTITY) as pi:
        _load_pool(pc, tensors, offs, dtype)
        _load_pool(pi, tensors, offs, dtype)
        for (nm, Wm), off, (N, K) in zip(tensors, offs, shapes):
            for batch in batches:
                X = gen.synth(seed + 100, batch, (batch, K), dtype, kind=gen.KIND_NORMAL)
                dX = _dev(X, dtype)
                yc, yi = torch.zeros(batch, N, dtype=dX.dtype, device="cuda"), torch.zeros(batch, N, dtype=dX.dtype, device="cuda")
                w = C.cloak_tensor(off, N, K, dt, C.CLOAK_ROWMAJOR)
                C.cloak_gemv(pc.h, w, dX, yc, batch)
                C.cloak_gemv(pi.h, w, dX, yi, batch)
                assert torch.equal(yc, yi)                                   # exact pin: same kernel, only addresses differ
                check_linear(yc.float().cpu().numpy(), X, Wm, dtype, f"gemv:{N}x{K}:b{batch}", TOL[dtype])


def test_gemv_closed_forms_through_the_table():
    """W = I gives Y = X; W = ones gives row sums -- read through a shuffled pool."""
    block, page, key, n = 4096, 65536, 0x1234, 256
    eye = np.eye(n, dtype=np.float32)
    ones = np.ones((n, n), dtype=np.float32)
    offs, total = C.cloak_arena_plan(key, [n * n * 4, n * n * 4], block)
    with Pool(total, block, page, key) as p:
        _load_pool(p, [("eye", eye), ("ones", ones)], offs, "f32")
        x = torch.randn(2, n, device="cuda")
        y = torch.zeros(2, n, device="cuda")
        C.cloak_gemv(p.h, C.cloak_tensor(offs[0], n, n, C.CLOAK_F32, C.CLOAK_ROWMAJOR), x, y, 2)
        assert torch.equal(x, y)
        C.cloak_gemv(p.h, C.cloak_tensor(offs[1], n, n, C.CLOAK_F32, C.CLOAK_ROWMAJOR), x, y, 2)
        assert torch.allclose(y, x.double().sum(dim=1, keepdim=True).float().expand(2, n), rtol=1e-5, atol=1e-5)
    # bf16: W = I exactly representable; x in bf16 comes back unchanged
    eyeb = O.f32_to_bf16_bits(eye)
    offs, total = C.cloak_arena_plan(key, [n * n * 2], block)
    with Pool(total, block, page, key) as p:
        _load_pool(p, [("eye", eyeb)], offs, "bf16")
        x = torch.randn(5, n, device="cuda").bfloat16()
        y = torch.zeros(5, n, device="cuda", dtype=torch.bfloat16)
        C.cloak_gemv(p.h, C.cloak_tensor(offs[0], n, n, C.CLOAK_BF16, C.CLOAK_ROWMAJOR), x, y, 5)
        assert torch.equal(x, y)


def test_gemv_host_entry_point():
    block, page, key, N, K = 65536, 2 << 20, 0x1234, 512, 1024
    Wm = gen.synth(1, 0, (N, K), "bf16")
    X = gen.synth(2, 0, (4, K), "bf16", kind=gen.KIND_NORMAL)
    with Pool(N * K * 2, block, page, key) as p:
        _load_pool(p, [("w", Wm)], [0], "bf16")
        hx = torch.from_numpy(X.view(np.int16).copy()).pin_memory()
        hy = torch.zeros(4, N, dtype=torch.int16).pin_memory()
        C.cloak_gemv_host(p.h, C.cloak_tensor(0, N, K, C.CLOAK_BF16, C.CLOAK_ROWMAJOR), hx, hy, 4)
        got = O.bf16_bits_to_f32(hy.numpy().view(np.uint16))
        check_linear(got, X, Wm, "bf16", f"gemv_host:{N}x{K}:b4", TOL["bf16"])
        # the chain form: several independent ops, host x / y, one synchronisation; equals the single host calls bit for bit
        hy2 = [torch.zeros(4, N, dtype=torch.int16).pin_memory() for _ in range(3)]
        w = C.cloak_tensor(0, N, K, C.CLOAK_BF16, C.CLOAK_ROWMAJOR)
        C.cloak_gemv_chain_host(p.h, [(w, hx, y, 0) for y in hy2], 4)
        assert all(torch.equal(y, hy) for y in hy2)
        with pytest.raises(C.CloakError) as ei:                       # dependent ops have no host form
            C.cloak_gemv_chain_host(p.h, [(w, hx, hy2[0], 0), (w, hx, hy2[1], 1)], 4)
        assert ei.value.status == C.CLOAK_ERR_INVALID


def test_cfg0_mlp_end_to_end_permuted_and_cloaked():
    """cfg0: permute -> shuffle -> three GEMVs + silu*up; equals the unpermuted MLP of the oracle (fp32 tol)."""
    c = gen.CONFIGS[0]
    H, I, key, block, page = c["hidden"], c["inter"], c["key"], c["block"], c["page"]
    gate, up, down = (gen.synth(c["seed"], i, s, "f32") for i, s in enumerate([(I, H), (I, H), (H, I)]))
    x = gen.synth(c["seed"], 10, (1, H), "f32", kind=gen.KIND_NORMAL)
    dg, du, dd = (torch.from_numpy(a.copy()).cuda() for a in (gate, up, down))
    pg, pu, pd = torch.empty_like(dg), torch.empty_like(du), torch.empty_like(dd)
    sh = C.cloak_block_shape(H, I, 0, 0, 0, C.CLOAK_F32, 0)
    C.cloak_permute_mlp_heads(key, sh, gate=dg, up=du, down=dd, gate_o=pg, up_o=pu, down_o=pd)
    offs, total = C.cloak_arena_plan(key, [4 * H * I] * 3, block)
    assert total == 3 << 20
    with Pool(total, block, page, key) as p:
        assert p.info["npages"] == 48
        for t, o in zip((pg, pu, pd), offs):
            C.cloak_shuffle(p.h, t, o, t.numel() * 4)
        dx = torch.from_numpy(x.copy()).cuda()
        yg, yu = torch.empty(1, I, device="cuda"), torch.empty(1, I, device="cuda")
        C.cloak_gemv(p.h, C.cloak_tensor(offs[0], I, H, C.CLOAK_F32, C.CLOAK_ROWMAJOR), dx, yg, 1)
        C.cloak_gemv(p.h, C.cloak_tensor(offs[1], I, H, C.CLOAK_F32, C.CLOAK_ROWMAJOR), dx, yu, 1)
        # the permuted gate output is the unpermuted one gathered by pi (the paper-level invariant, O9)
        pi = O.mlp_perm(key, 0, I).astype(np.int64)
        ref_g = O.linear_f64(x, gate)
        assert O.err_normwise(yg.cpu().numpy(), ref_g[:, pi]) <= TOL["f32"]
        act = torch.empty(1, I, device="cuda")
        C.cloak_silu_mul(yg, yu, act, I, C.CLOAK_F32)
        y = torch.empty(1, H, device="cuda")
        C.cloak_gemv(p.h, C.cloak_tensor(offs[2], H, I, C.CLOAK_F32, C.CLOAK_ROWMAJOR), act, y, 1)
        ref = O.mlp_f64(x, gate, up, down)                         # the UNpermuted MLP
        assert O.err_normwise(y.cpu().numpy(), ref) <= TOL["f32"]     # "GEMV and MLP err <= 1e-5 (fp32)"


# ------------------------------------------------------------------ S6 as one launch: cloak_gemv_chain
CHAIN_CASES = [
    # hidden, inter, n_q, n_kv, d, block, batches
    (256, 768, 4, 2, 64, 4096, [1, 5, 16]),             # small: 512 B / 1.5 KiB rows, several chunk sizes in one chain
    (1024, 3584, 8, 2, 128, 65536, [1, 4, 9]),          # 2 KiB and 7 KiB rows: two launch groups
    (4096, 14336, 32, 8, 128, 65536, [1, 16]),          # cfg1's layer: 4 KiB chunks, every CTA's range cut twice
]


@pytest.mark.parametrize("H,I,n_q,n_kv,d,block,batches", CHAIN_CASES)
def test_gemv_chain_layer_vs_single_calls_and_oracle(H, I, n_q, n_kv, d, block, batches):
    """One decoder layer's projections as ONE chain (q,k,v | o | gate,up | down with the fused silu*up input):
    bit-identical to the call-by-call path (cloak_gemv + cloak_silu_mul), bit-identical between the cloaked and
    the identity-table pool, within tolerance of the fp64 oracle (linear_f64 / mlp_f64), and repeatable."""
    key, seed, page = 0x1234, 1, 2 << 20 if block >= 65536 else 65536
    shapes = gen.layer_shapes(H, I, n_q, n_kv, d)
    Ws = {nm: gen.synth(seed, i, shp, "bf16") for i, (nm, shp) in enumerate(shapes)}
    sizes = [2 * n * k for _, (n, k) in shapes]
    offs, total = C.cloak_arena_plan(key, sizes, block)
    off = {nm: o for (nm, _), o in zip(shapes, offs)}
    with Pool(total, block, page, key) as pc, Pool(total, block, page, key, C.CLOAK_POOL_IDENTITY) as pi:
        for p in (pc, pi):
            _load_pool(p, [(nm, Ws[nm]) for nm, _ in shapes], offs, "bf16")
        T = {nm: C.cloak_tensor(off[nm], shp[0], shp[1], C.CLOAK_BF16, C.CLOAK_ROWMAJOR) for nm, shp in shapes}
        for batch in batches:
            xh = gen.synth(seed + 100, batch, (batch, H), "bf16", kind=gen.KIND_NORMAL)
            xa = gen.synth(seed + 200, batch, (batch, n_q * d), "bf16", kind=gen.KIND_NORMAL)
            dxh, dxa = bf16_dev_from_bits(xh), bf16_dev_from_bits(xa)

            def outputs():
                y = {nm: torch.zeros(batch, shp[0], dtype=torch.bfloat16, device="cuda") for nm, shp in shapes}
                y["act"] = torch.zeros(batch, I, dtype=torch.bfloat16, device="cuda")
                return y

            def run_chain(pool, y):
                ops = [(T["q"], dxh, y["q"], 0), (T["k"], dxh, y["k"], 0), (T["v"], dxh, y["v"], 0),
                       (T["o"], dxa, y["o"], 0), (T["gate"], dxh, y["gate"], 0),
                       (T["up"], dxh, y["up"], 0, y["gate"], y["act"]), (T["down"], y["act"], y["down"], 1)]
                C.cloak_gemv_chain(pool.h, ops, batch)

            yc, yi, ys, yr = outputs(), outputs(), outputs(), outputs()
            run_chain(pc, yc)
            run_chain(pi, yi)
            for nm in ("q", "k", "v", "gate", "up"):                       # call by call
                C.cloak_gemv(pc.h, T[nm], dxh, ys[nm], batch)
            C.cloak_gemv(pc.h, T["o"], dxa, ys["o"], batch)
            C.cloak_silu_mul(ys["gate"], ys["up"], ys["act"], batch * I, C.CLOAK_BF16)
            C.cloak_gemv(pc.h, T["down"], ys["act"], ys["down"], batch)
            run_chain(pc, yr)                                              # counters and barriers self-reset
            torch.cuda.synchronize()
            for nm in yc:
                assert torch.equal(yc[nm], yi[nm]), (nm, batch, "cloaked vs identity")
                assert torch.equal(yc[nm], ys[nm]), (nm, batch, "chain vs single calls")
                assert torch.equal(yc[nm], yr[nm]), (nm, batch, "second launch")
            for nm in ("q", "k", "v", "gate", "up"):
                check_linear(yc[nm].float().cpu().numpy(), xh, Ws[nm], "bf16", f"gemv_chain:H{H}:{nm}:b{batch}", TOL["bf16"])
            check_linear(yc["o"].float().cpu().numpy(), xa, Ws["o"], "bf16", f"gemv_chain:H{H}:o:b{batch}", TOL["bf16"])
            ref = O.mlp_f64(xh, Ws["gate"], Ws["up"], Ws["down"])           # fp64 all the way, no bf16 intermediates
            assert O.err_normwise(yc["down"].float().cpu().numpy(), ref) <= TOL["bf16"], (batch,)


def test_two_pools_two_streams_first_use_captured_without_warmup():
    """cloak.h, stream and scratch rules: no compute call synchronises the device or calls the driver's allocator; the
    pool's scratch exists from cloak_pool_create on (grown beforehand with cloak_pool_reserve_workspace where a GEMM needs
    more), so the FIRST use of a pool can be captured into a CUDA graph with no warm-up; two pools serve two non-blocking
    streams at the same time (the GEMV chains are cooperative launches: both grids cannot be resident at once, and the
    driver runs one after the other instead of leaving them spinning for each other's SMs)."""
    seed, block, page, H, I, bv, bm = 5, 65536, 2 << 20, 1024, 2048, 4, 64
    shapes = [("gate", (I, H)), ("up", (I, H)), ("down", (H, I))]
    Ws = {nm: gen.synth(seed, i, shp, "bf16") for i, (nm, shp) in enumerate(shapes)}
    sizes = [2 * n * k for _, (n, k) in shapes] * 2                       # ROWMAJOR copies, then TILE128 copies
    xv = gen.synth(seed + 100, 0, (bv, H), "bf16", kind=gen.KIND_NORMAL)
    xm = gen.synth(seed + 100, 1, (bm, H), "bf16", kind=gen.KIND_NORMAL)
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    pools, graphs, outs = [], [], []
    try:
        for key, st in zip((0x1234, 0x5678), streams):
            offs, total = C.cloak_arena_plan(key, sizes, block)
            p = Pool(total, block, page, key)
            pools.append(p)
            with torch.cuda.stream(st):
                dxv, dxm = bf16_dev_from_bits(xv), bf16_dev_from_bits(xm)
                for (nm, (n, k)), o, ot in zip(shapes, offs[:3], offs[3:]):
                    dW = bf16_dev_from_bits(Ws[nm])
                    C.cloak_shuffle(p.h, dW, o, dW.numel() * 2)
                    til = torch.empty_like(dW)
                    C.cloak_to_tile128(dW, til, n, k, C.CLOAK_BF16)
                    C.cloak_shuffle(p.h, til, ot, til.numel() * 2)
                T = {nm: C.cloak_tensor(o, n, k, C.CLOAK_BF16, C.CLOAK_ROWMAJOR) for (nm, (n, k)), o in zip(shapes, offs[:3])}
                Tt = {nm: C.cloak_tensor(o, n, k, C.CLOAK_BF16, C.CLOAK_TILE128) for (nm, (n, k)), o in zip(shapes, offs[3:])}
                y = {nm: torch.zeros(bv, n, dtype=torch.bfloat16, device="cuda") for nm, (n, k) in shapes}
                act = torch.zeros(bv, I, dtype=torch.bfloat16, device="cuda")
                yg = {nm: torch.zeros(bm, Tt[nm].N, dtype=torch.bfloat16, device="cuda") for nm in ("gate", "up")}
                vops = C.cloak_gemv_ops([(T["gate"], dxv, y["gate"], 0), (T["up"], dxv, y["up"], 0, y["gate"], act),
                                         (T["down"], act, y["down"], 1)])
                mops = C.cloak_gemm_ops([(Tt["gate"], dxm, yg["gate"]), (Tt["up"], dxm, yg["up"])])
                need = max(C.cloak_gemv_chain_scratch_bytes(p.h, vops, bv), C.cloak_gemm_chain_scratch_bytes(p.h, mops, bm))
                assert need > 0
                C.cloak_pool_reserve_workspace(p.h, need)                  # load time; synchronous
                st.synchronize()
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=st):                       # the pool's very first compute calls, captured
                    C.cloak_gemv_chain(p.h, vops, bv)
                    C.cloak_gemm_chain(p.h, mops, bm)
                graphs.append(g)
                outs.append((y, yg, vops, mops, dxv, dxm, act))
        for rep in range(3):                                               # both graphs in flight on their own streams
            for g, st in zip(graphs, streams):
                with torch.cuda.stream(st):
                    g.replay()
        torch.cuda.synchronize()
        for y, yg, *_ in outs:
            for nm in ("gate", "up"):
                check_linear(y[nm].float().cpu().numpy(), xv, Ws[nm], "bf16", f"two_streams:gemv:{nm}", TOL["bf16"])
                check_linear(yg[nm].float().cpu().numpy(), xm, Ws[nm], "bf16", f"two_streams:gemm:{nm}", TOL["bf16"])
            err = O.err_normwise(y["down"].float().cpu().numpy(), O.mlp_f64(xv, Ws["gate"], Ws["up"], Ws["down"]))
            assert err <= TOL["bf16"], err
        assert all(torch.equal(outs[0][0][nm], outs[1][0][nm]) for nm in outs[0][0])      # two keys, one function
        # a call that needs more scratch than the pool has fails inside a capture instead of allocating there ...
        p, st = pools[1], streams[1]                                      # (T, Tt hold the offsets of the last pool built)
        big = torch.zeros(256, Tt["gate"].N, dtype=torch.bfloat16, device="cuda")
        xbig = torch.zeros(256, H, dtype=torch.bfloat16, device="cuda")
        more = C.cloak_gemm_chain_scratch_bytes(p.h, [(Tt["gate"], xbig, big)] * 16, 256)
        if more > 16 << 20:
            g = torch.cuda.CUDAGraph()
            with pytest.raises(C.CloakError) as ei:
                with torch.cuda.graph(g, stream=st):
                    C.cloak_gemm_chain(p.h, [(Tt["gate"], xbig, big)] * 16, 256)
            assert ei.value.status == C.CLOAK_ERR_INVALID and "reserve" in str(ei.value)
            # ... and grows in stream order outside one, on a non-blocking side stream, with correct results afterwards
            with torch.cuda.stream(st):
                y1 = torch.zeros(bm, Tt["gate"].N, dtype=torch.bfloat16, device="cuda")
                C.cloak_gemm_chain(p.h, [(Tt["gate"], xbig, big)] * 16, 256)
                C.cloak_gemm(p.h, Tt["gate"], outs[1][5], y1, bm)
            st.synchronize()
            check_linear(y1.float().cpu().numpy(), xm, Ws["gate"], "bf16", "two_streams:after_growth", TOL["bf16"])
    finally:
        torch.cuda.synchronize()
        del graphs
        for p in pools:
            p.close()


def test_gemv_chain_argument_checks():
    with Pool(1 << 20, 4096, 65536, 0x1234) as p:
        x = torch.zeros(1, 256, dtype=torch.bfloat16, device="cuda")
        y = torch.zeros(1, 64, dtype=torch.bfloat16, device="cuda")
        good = C.cloak_tensor(0, 64, 256, C.CLOAK_BF16, C.CLOAK_ROWMAJOR)
        C.cloak_gemv_chain(p.h, [(good, x, y, 0)], 1)
        for bad, status in ((C.cloak_tensor(0, 64, 64, C.CLOAK_BF16, C.CLOAK_ROWMAJOR), C.CLOAK_ERR_UNSUPPORTED),   # K % 256
                            (C.cloak_tensor(0, 64, 256, C.CLOAK_F32, C.CLOAK_ROWMAJOR), C.CLOAK_ERR_UNSUPPORTED),
                            (C.cloak_tensor(4096 * 255, 64, 256, C.CLOAK_BF16, C.CLOAK_ROWMAJOR), C.CLOAK_ERR_INVALID)):
            with pytest.raises(C.CloakError) as e:
                C.cloak_gemv_chain(p.h, [(good, x, y, 0), (bad, x, y, 0)], 1)
            assert e.value.status == status
        with pytest.raises(C.CloakError):
            C.cloak_gemv_chain(p.h, [(good, x, y, 0)], 17)
        with pytest.raises(C.CloakError):                                   # d_gate without d_act
            C.cloak_gemv_chain(p.h, [(good, x, y, 0, y, None)], 1)
        torch.cuda.synchronize()


# ------------------------------------------------------------------ S7 cloaked GEMM (tcgen05, TILE128)
GEMM_CASES = [
    # block, shapes [(N, K)], batches
    (32768, [(128, 128), (256, 384)], [16, 32]),                        # one tile; several tiles, one tile per block
    (65536, [(1024, 5120), (5120, 1024)], [32, 128]),                   # cfg3's k/v shape and a tall one; stream-K cuts
    (65536, [(384, 640)], [48, 256]),                                   # odd tile counts, widest batch
    (2 << 20, [(512, 512)], [64]),                                      # block == page
    (65536, [(1024, 2048), (384, 640)], [1, 4, 13, 200]),              # batches that are not multiples of 16 (zero-padded MMA columns)
]


@pytest.mark.parametrize("block,shapes,batches", GEMM_CASES)
def test_gemm_vs_oracle_and_identity_bit_identical(block, shapes, batches):
    key, seed, page = 0x1234, 3, 2 << 20
    tensors = [(f"t{i}", gen.synth(seed, i, shp, "bf16")) for i, shp in enumerate(shapes)]
    sizes = [a.size * 2 for _, a in tensors]
    offs, total = C.cloak_arena_plan(key, sizes, block)
    with Pool(total, block, page, key) as pc, Pool(total, block, page, key, C.CLOAK_POOL_IDENTITY) as pi:
        for (nm, Wm), off in zip(tensors, offs):
            N, K = Wm.shape
            src = bf16_dev_from_bits(Wm)
            til = torch.empty(N * K, dtype=torch.bfloat16, device="cuda")
            C.cloak_to_tile128(src, til, N, K, C.CLOAK_BF16)                 # O0 stage (2): storage layout
            assert np.array_equal(bits_from_bf16_dev(til), O.to_tile128(Wm))
            for p in (pc, pi):
                C.cloak_shuffle(p.h, til, off, N * K * 2)
        for (nm, Wm), off in zip(tensors, offs):
            N, K = Wm.shape
            w = C.cloak_tensor(off, N, K, C.CLOAK_BF16, C.CLOAK_TILE128)
            for batch in batches:
                X = gen.synth(seed + 100, batch, (batch, K), "bf16", kind=gen.KIND_NORMAL)
                dX = bf16_dev_from_bits(X)
                yc = torch.zeros(batch, N, dtype=torch.bfloat16, device="cuda")
                yi = torch.zeros_like(yc)
                C.cloak_gemm(pc.h, w, dX, yc, batch)
                C.cloak_gemm(pi.h, w, dX, yi, batch)
                torch.cuda.synchronize()
                assert torch.equal(yc, yi)
                check_linear(yc.float().cpu().numpy(), X, Wm, "bf16", f"gemm:{N}x{K}:b{batch}", TOL["bf16"])
                yc2 = torch.zeros_like(yc)                                   # second launch: counters self-reset
                C.cloak_gemm(pc.h, w, dX, yc2, batch)
                assert torch.equal(yc, yc2)


@pytest.mark.parametrize("batch", [32, 128])
def test_gemm_chain_equals_single_calls(batch):
    """cloak_gemm_chain: 20 ops of mixed shapes (two launches of <= 16 ops): bit-identical on the cloaked and the
    identity-table pool, repeatable; equal to cloak_gemm op by op up to the fp32 summation order (a chain cuts K where
    its ranges fall); every op against the fp64 oracle."""
    key, seed, block, page = 0x1234, 3, 65536, 2 << 20
    shapes = [(1024, 5120), (5120, 1024), (384, 640), (128, 128), (2560, 2560)] * 4
    Ws = [gen.synth(seed, i, shp, "bf16") for i, shp in enumerate(shapes[:5])]
    sizes = [2 * n * k for n, k in shapes]
    offs, total = C.cloak_arena_plan(key, sizes, block)
    with Pool(total, block, page, key) as pc, Pool(total, block, page, key, C.CLOAK_POOL_IDENTITY) as pi:
        for i, ((n, k), off) in enumerate(zip(shapes, offs)):
            src = bf16_dev_from_bits(Ws[i % 5])
            til = torch.empty(n * k, dtype=torch.bfloat16, device="cuda")
            C.cloak_to_tile128(src, til, n, k, C.CLOAK_BF16)
            for p in (pc, pi):
                C.cloak_shuffle(p.h, til, off, n * k * 2)
        X = {k: gen.synth(seed + 100, k, (batch, k), "bf16", kind=gen.KIND_NORMAL) for k in {k for _, k in shapes}}
        dX = {k: bf16_dev_from_bits(v) for k, v in X.items()}
        T = [C.cloak_tensor(off, n, k, C.CLOAK_BF16, C.CLOAK_TILE128) for (n, k), off in zip(shapes, offs)]

        def outs():
            return [torch.zeros(batch, n, dtype=torch.bfloat16, device="cuda") for n, _ in shapes]
        yc, yi, ys, yr = outs(), outs(), outs(), outs()
        C.cloak_gemm_chain(pc.h, [(T[i], dX[shapes[i][1]], yc[i]) for i in range(len(shapes))], batch)
        C.cloak_gemm_chain(pi.h, [(T[i], dX[shapes[i][1]], yi[i]) for i in range(len(shapes))], batch)
        for i in range(len(shapes)):
            C.cloak_gemm(pc.h, T[i], dX[shapes[i][1]], ys[i], batch)
        C.cloak_gemm_chain(pc.h, [(T[i], dX[shapes[i][1]], yr[i]) for i in range(len(shapes))], batch)
        torch.cuda.synchronize()
        for i in range(len(shapes)):
            assert torch.equal(yc[i], yi[i]) and torch.equal(yc[i], yr[i]), i
            d = (yc[i].float() - ys[i].float()).norm() / ys[i].float().norm()
            assert d <= 4e-3, (i, float(d))                                  # bf16 rounding of two fp32 summation orders
        for i in range(len(shapes)):
            check_linear(yc[i].float().cpu().numpy(), X[shapes[i][1]], Ws[i % 5], "bf16", f"gemm_chain:b{batch}:op{i}", TOL["bf16"])


@pytest.mark.parametrize("batch", [16, 32, 50, 64, 128])
def test_gemm_row_groups(batch):
    """cloak_set_gemm_engine: tile rows in pairs (3; 0 = where the launch is large enough), singly (1), or in fours (2) share each X tile -- two or four accumulators
    per segment in TMEM, units of two / four weight tiles, tickets per row.  Under each setting: every op against the fp64
    oracle, the chain repeatable bit for bit and identical on the identity-table pool; single calls too.  Shapes with 2, 4, 6, 8
    and 20 tile rows (6 is not a multiple of four: the launch falls back to pairs), one launch that mixes in an odd row count
    (falls back to single rows)."""
    key, seed, block, page = 0x1234, 13, 65536, 2 << 20
    shapes = [(1024, 2560), (512, 1280), (256, 5120), (2560, 640), (768, 1024)]
    Ws = [gen.synth(seed, i, shp, "bf16") for i, shp in enumerate(shapes)] + [gen.synth(seed, 9, (384, 640), "bf16")]
    all_shapes = shapes + [(384, 640)]
    offs, total = C.cloak_arena_plan(key, [2 * n * k for n, k in all_shapes], block)
    try:
        with Pool(total, block, page, key) as pc, Pool(total, block, page, key, C.CLOAK_POOL_IDENTITY) as pi:
            for (n, k), off, Wm in zip(all_shapes, offs, Ws):
                til = torch.empty(n * k, dtype=torch.bfloat16, device="cuda")
                C.cloak_to_tile128(bf16_dev_from_bits(Wm), til, n, k, C.CLOAK_BF16)
                for p in (pc, pi):
                    C.cloak_shuffle(p.h, til, off, n * k * 2)
            T = [C.cloak_tensor(o, n, k, C.CLOAK_BF16, C.CLOAK_TILE128) for (n, k), o in zip(all_shapes, offs)]
            X = {k: gen.synth(seed + 50, k, (batch, k), "bf16", kind=gen.KIND_NORMAL) for k in {k for _, k in all_shapes}}
            dX = {k: bf16_dev_from_bits(v) for k, v in X.items()}

            def run(pool, idx, single=False):
                ys = [torch.zeros(batch, all_shapes[w][0], dtype=torch.bfloat16, device="cuda") for w in idx]
                if single:
                    for w, y in zip(idx, ys):
                        C.cloak_gemm(pool.h, T[w], dX[all_shapes[w][1]], y, batch)
                else:
                    C.cloak_gemm_chain(pool.h, [(T[w], dX[all_shapes[w][1]], y) for w, y in zip(idx, ys)], batch)
                torch.cuda.synchronize()
                return ys
            for eng in (0, 1, 2, 3):
                C.cloak_set_gemm_engine(eng)
                for idx in ([0, 1, 2, 3, 0, 2], [0, 1, 2, 3, 4], [0, 5, 3]):          # fours possible | pairs at most | single rows
                    a, b, c = run(pc, idx), run(pc, idx), run(pi, idx)
                    s1 = run(pc, idx, single=True)
                    for j, w in enumerate(idx):
                        assert torch.equal(a[j], b[j]) and torch.equal(a[j], c[j]), (eng, idx, j)
                        check_linear(a[j].float().cpu().numpy(), X[all_shapes[w][1]], Ws[w], "bf16", f"gemm_groups:b{batch}:e{eng}:op{w}", TOL["bf16"])
                        check_linear(s1[j].float().cpu().numpy(), X[all_shapes[w][1]], Ws[w], "bf16", f"gemm_groups_single:b{batch}:e{eng}:op{w}", TOL["bf16"])
    finally:
        C.cloak_set_gemm_engine(0)


def test_gemm_argument_checks():
    with Pool(1 << 20, 4096, 65536, 1) as p:
        x = torch.zeros(32, 128, dtype=torch.bfloat16, device="cuda")
        y = torch.zeros(32, 128, dtype=torch.bfloat16, device="cuda")
        for w, batch, st in [
            (C.cloak_tensor(0, 128, 128, C.CLOAK_BF16, C.CLOAK_TILE128), 32, C.CLOAK_ERR_UNSUPPORTED),   # 4 KiB blocks
            (C.cloak_tensor(0, 128, 128, C.CLOAK_BF16, C.CLOAK_ROWMAJOR), 32, C.CLOAK_ERR_UNSUPPORTED),
            (C.cloak_tensor(0, 128, 128, C.CLOAK_BF16, C.CLOAK_TILE128), 0, C.CLOAK_ERR_INVALID),
            (C.cloak_tensor(0, 128, 128, C.CLOAK_BF16, C.CLOAK_TILE128), 257, C.CLOAK_ERR_INVALID),
            (C.cloak_tensor(0, 100, 128, C.CLOAK_BF16, C.CLOAK_TILE128), 32, C.CLOAK_ERR_ALIGN),
        ]:
            with pytest.raises(C.CloakError) as ei:
                C.cloak_gemm(p.h, w, x, y, batch)
            assert ei.value.status == st


@pytest.mark.parametrize("batch", [32, 128, 208])
def test_gemm_schedules_agree(batch):
    """cloak_set_gemm_schedule: the chunk grid (static share, dynamic chunk cap) decides where K is split.  Under every
    setting -- all static, the default, nearly all dynamic with small pieces (many contributors per tile row) -- a chain
    of 10 ops is repeatable bit for bit (which CTA draws which chunk varies from launch to launch), the same on the
    cloaked and the identity-table pool, and within the bf16 tolerance of the fp64 oracle."""
    key, seed, block, page = 0x1234, 3, 65536, 2 << 20
    shapes = [(2560, 2560), (1024, 5120), (5120, 1024), (384, 640), (128, 128)] * 2
    Ws = [gen.synth(seed, i, shp, "bf16") for i, shp in enumerate(shapes[:5])]
    sizes = [2 * n * k for n, k in shapes]
    offs, total = C.cloak_arena_plan(key, sizes, block)
    try:
        with Pool(total, block, page, key) as pc, Pool(total, block, page, key, C.CLOAK_POOL_IDENTITY) as pi:
            for i, ((n, k), off) in enumerate(zip(shapes, offs)):
                til = torch.empty(n * k, dtype=torch.bfloat16, device="cuda")
                C.cloak_to_tile128(bf16_dev_from_bits(Ws[i % 5]), til, n, k, C.CLOAK_BF16)
                for p in (pc, pi):
                    C.cloak_shuffle(p.h, til, off, n * k * 2)
            X = {k: gen.synth(seed + 100, k, (batch, k), "bf16", kind=gen.KIND_NORMAL) for k in {k for _, k in shapes}}
            dX = {k: bf16_dev_from_bits(v) for k, v in X.items()}
            T = [C.cloak_tensor(off, n, k, C.CLOAK_BF16, C.CLOAK_TILE128) for (n, k), off in zip(shapes, offs)]
            refs = [O.linear_f64(X[k], Ws[i]) for i, (n, k) in enumerate(shapes[:5])]

            def run(pool):
                ys = [torch.zeros(batch, n, dtype=torch.bfloat16, device="cuda") for n, _ in shapes]
                C.cloak_gemm_chain(pool.h, [(T[i], dX[shapes[i][1]], ys[i]) for i in range(len(shapes))], batch)
                torch.cuda.synchronize()
                return ys
            for sched in ((100, 0), (75, 0), (10, 3), (0, 7), (50, 64)):
                C.cloak_set_gemm_schedule(*sched)
                a, b, c = run(pc), run(pc), run(pi)
                for i in range(len(shapes)):
                    assert torch.equal(a[i], b[i]) and torch.equal(a[i], c[i]), (sched, i)
                    check_linear(a[i].float().cpu().numpy(), X[shapes[i][1]], Ws[i % 5], "bf16",
                                 f"gemm_sched:b{batch}:{sched[0]}/{sched[1]}:op{i}", TOL["bf16"])
    finally:
        C.cloak_set_gemm_schedule(75, 0)
    for bad in ((-1, 0), (101, 0), (75, -1), (75, 5000)):
        with pytest.raises(C.CloakError) as ei:
            C.cloak_set_gemm_schedule(*bad)
        assert ei.value.status == C.CLOAK_ERR_INVALID


# ------------------------------------------------------------------ errors
def test_error_codes_on_device():
    with Pool(1 << 20, 4096, 65536, 1) as p:
        buf = dev_bytes(8192)
        for fn, args, st in [
            (C.cloak_shuffle, (p.h, buf, 100, 4096), C.CLOAK_ERR_ALIGN),
            (C.cloak_shuffle, (p.h, buf, 0, 100), C.CLOAK_ERR_ALIGN),
            (C.cloak_shuffle, (p.h, buf, 1 << 20, 4096), C.CLOAK_ERR_INVALID),
            (C.cloak_unshuffle, (p.h, None, 0, 4096), C.CLOAK_ERR_INVALID),
            (C.cloak_relayout, (p.h, p.h), C.CLOAK_ERR_INVALID),
        ]:
            with pytest.raises(C.CloakError) as ei:
                fn(*args)
            assert ei.value.status == st
        x = torch.zeros(1, 256, device="cuda")
        with pytest.raises(C.CloakError) as ei:
            C.cloak_gemv(p.h, C.cloak_tensor(0, 1024, 256, C.CLOAK_F32, C.CLOAK_ROWMAJOR), x, x, 17)
        assert ei.value.status == C.CLOAK_ERR_INVALID
        with pytest.raises(C.CloakError) as ei:
            C.cloak_gemv(p.h, C.cloak_tensor(0, 1024, 256, C.CLOAK_F32, C.CLOAK_TILE128), x, x, 1)
        assert ei.value.status == C.CLOAK_ERR_UNSUPPORTED
        with pytest.raises(C.CloakError) as ei:
            C.cloak_gemv(p.h, C.cloak_tensor(0, 1 << 20, 256, C.CLOAK_F32, C.CLOAK_ROWMAJOR), x, x, 1)
        assert ei.value.status == C.CLOAK_ERR_INVALID
        with pytest.raises(C.CloakError) as ei:                       # emulated pages cannot be re-mapped
            C.cloak_rekey_pages_begin(p.h, 2, 1)
        assert ei.value.status == C.CLOAK_ERR_UNSUPPORTED
        assert C.cloak_rekey_pages_step(p.h, 4) == 0                   # no re-key in progress: nothing left, no error
        C.cloak_pool_reserve_workspace(p.h, 1 << 20)                   # already there: a no-op
        C.cloak_pool_reserve_workspace(p.h, 40 << 20)                  # grows
    with Pool(8 << 20, 65536, 2 << 20, 1) as p, Pool(8 << 20, 65536, 2 << 20, 1, C.CLOAK_POOL_IDENTITY) as pi:
        with pytest.raises(C.CloakError) as ei:
            C.cloak_rekey_pages_begin(pi.h, 2, 1)
        assert ei.value.status == C.CLOAK_ERR_INVALID
        with pytest.raises(C.CloakError) as ei:
            C.cloak_rekey_pages_begin(p.h, 2, 65)
        assert ei.value.status == C.CLOAK_ERR_INVALID
        C.cloak_rekey_pages_begin(p.h, 2, 1)
        for call in (lambda: C.cloak_rekey_pages_begin(p.h, 3, 1), lambda: C.cloak_rekey_inplace(p.h, 3, 0)):
            with pytest.raises(C.CloakError) as ei:                   # one re-key at a time
                call()
            assert ei.value.status == C.CLOAK_ERR_INVALID
        # (the pool is destroyed with the re-key unfinished: its teardown must cope)


# ------------------------------------------------------------------ NEXT-4: mixture-of-experts layers
@pytest.mark.parametrize("E,H,I,dtype,layer", [(6, 64, 40, "f32", 0), (8, 256, 1000, "bf16", 3), (32, 2048, 768, "bf16", 47),
                                                  (5, 264, 4096, "bf16", 1), (3, 72, 4104, "bf16", 2), (7, 128, 8, "bf16", 9), (4, 64, 1000, "f32", 4)])
def test_permute_experts_bit_exact(E, H, I, dtype, layer):
    """cloak_permute_experts against the oracle: router rows and whole experts by eps, each expert's neurons by its own pi.
    bf16 with inter <= 4096 takes the batched path (one keygen launch for all experts, one row gather each for gate and up, one
    short-row column gather for down: ragged last row block at hidden = 264, the 8 KiB row limit at inter = 4096, one vector per
    row at inter = 8); inter = 4104 and f32 take the expert-by-expert path."""
    key, seed = 0x1234, 9
    router = gen.synth(seed, 0, (E, H), dtype)
    gate, up = gen.synth(seed, 1, (E, I, H), dtype), gen.synth(seed, 2, (E, I, H), dtype)
    down = gen.synth(seed, 3, (E, H, I), dtype)
    dev = [_dev(a, dtype) for a in (router, gate, up, down)]
    out = [torch.zeros_like(t) for t in dev]
    sh = C.cloak_moe_shape(H, I, E, C.CLOAK_F32 if dtype == "f32" else C.CLOAK_BF16, layer)
    C.cloak_permute_experts(key, sh, *dev, *out)
    eps = O.expert_perm(key, layer, E)
    pis = [O.expert_mlp_perm(key, layer, E, e, I) for e in range(E)]
    ref = O.permute_experts(router, gate, up, down, eps, pis)
    for o_, r_ in zip(out, ref):
        got = o_.cpu().numpy() if dtype == "f32" else bits_from_bf16_dev(o_)
        assert np.array_equal(got, r_)


def test_moe_decode_through_the_cloaked_pool_equals_the_unpermuted_moe():
    """Expert permutation -> block shuffle -> router GEMV + one cloak_gemv_chain over the selected experts (gate | up with
    the silu*up epilogue | down): equals the oracle's UNpermuted MoE forward (fp64) within the bf16 tolerance."""
    key, seed, layer, E, H, I, k, block, page = 0x1234, 4, 1, 8, 512, 256, 2, 65536, 2 << 20
    router = gen.synth(seed, 0, (E, H), "bf16", kind=gen.KIND_NORMAL)       # O(1) logits so that the top-k is well separated
    gate, up, down = gen.synth(seed, 1, (E, I, H), "bf16"), gen.synth(seed, 2, (E, I, H), "bf16"), gen.synth(seed, 3, (E, H, I), "bf16")
    dev = [bf16_dev_from_bits(a) for a in (router, gate, up, down)]
    prm = [torch.zeros_like(t) for t in dev]
    C.cloak_permute_experts(key, C.cloak_moe_shape(H, I, E, C.CLOAK_BF16, layer), *dev, *prm)
    eps = O.expert_perm(key, layer, E)
    new_of_old = {int(eps[en]): en for en in range(E)}
    # arena: padded router (16 rows at least for the GEMV), then gate_e, up_e, down_e of every (new) expert
    rpad = torch.zeros(16, H, dtype=torch.bfloat16, device="cuda")
    rpad[:E] = prm[0]
    sizes = [16 * H * 2] + [I * H * 2] * (3 * E)
    offs, total = C.cloak_arena_plan(key, sizes, block)
    with Pool(total, block, page, key) as p:
        C.cloak_shuffle(p.h, rpad, offs[0], rpad.numel() * 2)
        T = {}
        for en in range(E):
            for j, (nm, t, n, kk) in enumerate((("gate", prm[1], I, H), ("up", prm[2], I, H), ("down", prm[3], H, I))):
                o = offs[1 + 3 * en + j]
                C.cloak_shuffle(p.h, t[en], o, I * H * 2)
                T[nm, en] = C.cloak_tensor(o, n, kk, C.CLOAK_BF16, C.CLOAK_ROWMAJOR)
        for tok in range(3):
            x = gen.synth(seed + 100, tok, (1, H), "bf16", kind=gen.KIND_NORMAL)
            dx = bf16_dev_from_bits(x)
            logits_d = torch.zeros(1, 16, dtype=torch.bfloat16, device="cuda")
            C.cloak_gemv(p.h, C.cloak_tensor(offs[0], 16, H, C.CLOAK_BF16, C.CLOAK_ROWMAJOR), dx, logits_d, 1)
            ref_logits = O.linear_f64(x, router)[0]
            got_logits = logits_d.float().cpu().numpy()[0, :E]
            assert O.err_normwise(got_logits, ref_logits[eps.astype(np.int64)]) <= TOL["bf16"]      # logits move with the experts
            sel_old = O.topk_experts(ref_logits, k)                         # routing decided in fp64, then relabelled
            z = ref_logits[sel_old]
            w = np.exp(z - z.max())
            w /= w.sum()
            ys, ups, downs = [], [], []
            for i, e_old in enumerate(sel_old):
                en = new_of_old[e_old]
                yg, yu, act = (torch.zeros(1, I, dtype=torch.bfloat16, device="cuda") for _ in range(3))
                yd = torch.zeros(1, H, dtype=torch.bfloat16, device="cuda")
                ups += [(T["gate", en], dx, yg, 0), (T["up", en], dx, yu, 0, yg, act)]
                downs.append((T["down", en], act, yd, 1 if i == 0 else 2))      # all downs share one grid-wide arrival
                ys.append(yd)
            C.cloak_gemv_chain(p.h, ups + downs, 1)
            torch.cuda.synchronize()
            got = sum(wi * y.double().cpu().numpy() for wi, y in zip(w, ys))
            assert O.err_normwise(got, O.moe_f64(x, router, gate, up, down, k)) <= TOL["bf16"], tok


@pytest.mark.parametrize("batch,I", [(1, 256), (4, 256), (8, 512), (3, 512), (16, 256)])
def test_gemv_chain_fuses_small_ops_bit_identically(batch, I):
    """Ops whose rows are one chunk (the experts' projections of an MoE layer) are dealt out as ONE op per (shape, run) at
    batch <= 8 (gemv_stream.cu: fusion).  The fused launch must equal the unfused one (cloak_set_gemv_engine(4)) bit for
    bit, on cloaked and identity pools, for: an MoE-shaped layer (gate_e | up_e with the silu epilogue | down_e after them, an
    attention block and a router before, two layers back to back), experts listed gate, gate, .., up, up, .. instead, a gate
    taken from ANOTHER expert's projection (no fusion possible: must still be right), and a big op between the small ones;
    every down output against the fp64 oracle of silu(gate x) * (up x) through down."""
    key, seed, block, page = 0x1234, 31, 65536, 2 << 20
    H, E, Q = 512, 6, 1024          # rows of 1 KiB (gate / up) and 512 B (down, I = 256): one chunk each, downs in launches of their
                                    # own; I = 512: one chunk size for all three -- the fused downs wait for the fused ups INSIDE a launch
    shapes = {"q": (Q, H), "o": (H, Q), "router": (16, H), "big": (1024, 4096)}
    for e in range(E):
        shapes.update({f"gate{e}": (I, H), f"up{e}": (I, H), f"down{e}": (H, I)})
    names = list(shapes)
    Ws = {nm: gen.synth(seed, i, shapes[nm], "bf16") for i, nm in enumerate(names)}
    offs, total = C.cloak_arena_plan(key, [2 * n * k for n, k in shapes.values()], block)
    off = dict(zip(names, offs))
    try:
        with Pool(total, block, page, key) as pc, Pool(total, block, page, key, C.CLOAK_POOL_IDENTITY) as pi:
            _load_pool(pc, [(nm, Ws[nm]) for nm in names], offs, "bf16")
            _load_pool(pi, [(nm, Ws[nm]) for nm in names], offs, "bf16")
            T = {nm: C.cloak_tensor(off[nm], *shapes[nm], C.CLOAK_BF16, C.CLOAK_ROWMAJOR) for nm in names}
            Xh = gen.synth(seed + 1, 0, (batch, H), "bf16", kind=gen.KIND_NORMAL)
            Xq = gen.synth(seed + 1, 1, (batch, Q), "bf16", kind=gen.KIND_NORMAL)
            Xb = gen.synth(seed + 1, 2, (batch, 4096), "bf16", kind=gen.KIND_NORMAL)
            xh, xq, xb = bf16_dev_from_bits(Xh), bf16_dev_from_bits(Xq), bf16_dev_from_bits(Xb)
            z = lambda n: torch.zeros(batch, n, dtype=torch.bfloat16, device="cuda")      # noqa: E731

            def build(variant):
                ops, outs, downs_of = [], [], []
                for layer in range(2):
                    ops += [(T["q"], xh, z(Q), 0), (T["o"], xq, z(H), 0), (T["router"], xh, z(16), 0)]
                    sel = [0, 2, 3, 5] if layer == 0 else [1, 2, 4, 5]
                    g = {e: z(I) for e in sel}
                    u = {e: z(I) for e in sel}
                    act = {e: z(I) for e in sel}
                    d = {e: z(H) for e in sel}
                    if variant == "interleaved":
                        for e in sel:
                            ops += [(T[f"gate{e}"], xh, g[e], 0), (T[f"up{e}"], xh, u[e], 0, g[e], act[e])]
                    elif variant == "grouped":
                        ops += [(T[f"gate{e}"], xh, g[e], 0) for e in sel] + [(T[f"up{e}"], xh, u[e], 0, g[e], act[e]) for e in sel]
                    elif variant == "big_between":
                        for i, e in enumerate(sel):
                            ops += [(T[f"gate{e}"], xh, g[e], 0)] + ([(T["big"], xb, z(1024), 0)] if i == 1 else []) + [(T[f"up{e}"], xh, u[e], 0, g[e], act[e])]
                    else:                           # "crossed": up_e's epilogue takes the gate of the NEXT expert's projection
                        for e in sel:
                            ops += [(T[f"gate{e}"], xh, g[e], 0)]
                        for i, e in enumerate(sel):
                            ops += [(T[f"up{e}"], xh, u[e], 0, g[sel[(i + 1) % len(sel)]], act[e])]
                    ops += [(T[f"down{e}"], act[e], d[e], 1 if i == 0 else 2) for i, e in enumerate(sel)]
                    downs_of.append((sel, d, variant))
                    outs += [t[e] for e in sel for t in (g, u, act, d)]
                outs += [op[2] for op in ops]
                return ops, outs, downs_of

            for variant in ("interleaved", "grouped", "big_between", "crossed"):
                res = {}
                for eng in (0, 4):
                    C.cloak_set_gemv_engine(eng)
                    for pool_name, pool in (("c", pc), ("i", pi)):
                        ops, outs, downs_of = build(variant)
                        C.cloak_gemv_chain(pool.h, ops, batch)
                        C.cloak_gemv_chain(pool.h, ops, batch)           # again over the same outputs: counters back at zero
                        torch.cuda.synchronize()
                        res[eng, pool_name] = (outs, downs_of)
                base = res[4, "c"][0]
                for k_, (outs, _) in res.items():
                    assert all(torch.equal(a_, b_) for a_, b_ in zip(outs, base)), (variant, k_)
                assert any(float(t.float().abs().sum()) > 0 for t in base)
                # the down outputs against the oracle
                for sel, d, var in res[0, "c"][1]:
                    for i, e in enumerate(sel):
                        ge = sel[(i + 1) % len(sel)] if var == "crossed" else e
                        ref = O.mlp_f64(Xh, Ws[f"gate{ge}"], Ws[f"up{e}"], Ws[f"down{e}"])       # O9, unrounded intermediates
                        assert O.err_normwise(d[e].double().cpu().numpy(), ref) <= TOL["bf16"], (variant, e)
    finally:
        C.cloak_set_gemv_engine(0)


@pytest.mark.parametrize("batch", [1, 8, 16])
def test_gemv_chain_helper_queue_wraps(batch):
    """The helper warp's 8-slot record queue under load: 48 ops in ONE launch, every op with cut row tiles (two or four chunks per
    row) and `after = 1` -- a publish, a tail and a report per op and CTA, a grid-wide wait before every op -- alternating between
    a generator vector and the previous op's output as input; twice over the same outputs (counters back at zero).  Equal to the
    same ops issued one cloak_gemv at a time, bit for bit; the ops fed by the generator vector also against the oracle."""
    key, seed, block, page = 0x1234, 41, 65536, 2 << 20
    shapes = [(2560, 2560), (2560, 5120), (5120, 2560)]            # 5 KiB and 10 KiB rows: 2.5 KiB chunks, kch = 2 / 4
    Ws = [gen.synth(seed, i, shp, "bf16") for i, shp in enumerate(shapes)]
    offs, total = C.cloak_arena_plan(key, [2 * n * k for n, k in shapes], block)
    with Pool(total, block, page, key) as p:
        _load_pool(p, [(f"w{i}", w) for i, w in enumerate(Ws)], offs, "bf16")
        T = [C.cloak_tensor(o, n, k, C.CLOAK_BF16, C.CLOAK_ROWMAJOR) for (n, k), o in zip(shapes, offs)]
        X = {k: gen.synth(seed + 1, k, (batch, k), "bf16", kind=gen.KIND_NORMAL) for k in (2560, 5120)}
        dX = {k: bf16_dev_from_bits(v) for k, v in X.items()}
        order = [0, 1, 2] * 16                                       # every third op (K = 2560) reads the output of the one before it (N = 2560)
        outs_c, outs_s, ops, singles = [], [], [], []
        for j, w in enumerate(order):
            n, k = shapes[w]
            yc, ys = torch.zeros(batch, n, dtype=torch.bfloat16, device="cuda"), torch.zeros(batch, n, dtype=torch.bfloat16, device="cuda")
            fresh = j % 3 != 2                                       # ops 2, 5, ..: X is the previous op's output
            xc = dX[k] if fresh else outs_c[j - 1]
            xs = dX[k] if fresh else outs_s[j - 1]
            ops.append((T[w], xc, yc, 1))
            singles.append((T[w], xs, ys, fresh))
            outs_c.append(yc)
            outs_s.append(ys)
        launches0 = C.cloak_launch_count()
        C.cloak_gemv_chain(p.h, ops, batch)
        assert C.cloak_launch_count() - launches0 == 1
        C.cloak_gemv_chain(p.h, ops, batch)
        for t, x, y, _ in singles:
            C.cloak_gemv(p.h, t, x, y, batch)
        torch.cuda.synchronize()
        for j in range(len(order)):
            assert torch.equal(outs_c[j], outs_s[j]), j
        for j in (0, 1, 3, 45, 46):
            assert singles[j][3]
            check_linear(outs_c[j].float().cpu().numpy(), X[shapes[order[j]][1]], Ws[order[j]], "bf16", f"gemv_chain_queue:b{batch}:op{j}", TOL["bf16"])


# ------------------------------------------------------------------ randomised chains (shapes, lengths, dependencies)
@pytest.mark.parametrize("seed", [0, 1, 2, 3, 10, 11, 12, 13, 14, 15, 16, 17])
def test_gemv_chain_random_lists_equal_single_calls(seed):
    """Random op lists (1..60 ops, rows of 512 B .. 28 KiB, N from 16 to 4 096, mixed chunk sizes -> several launches,
    random `after` 0/1/2 with real data dependencies, random gate epilogues): bit-identical to the same ops issued one
    cloak_gemv / cloak_silu_mul at a time, and every op fed by a generator vector against the fp64 oracle."""
    rng = np.random.default_rng(100 + seed)
    key, block, page = 0x1234, 65536, 2 << 20
    small = seed >= 10        # seeds >= 10: few tensors, rows of one chunk, batch <= 8 -- the launch planner fuses whatever it may
    batch = int(rng.choice([1, 3, 8] if small else [1, 3, 8, 9, 16]))
    n_w = 3 if small else 6
    shapes = [(int(rng.choice([16, 48, 256, 512] if small else [16, 48, 256, 1024, 4096])),
               int(rng.choice([256, 512, 1024, 2048] if small else [256, 512, 768, 2048, 3584, 14336]))) for _ in range(n_w)]
    Ws = [gen.synth(seed, i, shp, "bf16") for i, shp in enumerate(shapes)]
    offs, total = C.cloak_arena_plan(key, [2 * n * k for n, k in shapes], block)
    with Pool(total, block, page, key) as p:
        _load_pool(p, [(f"w{i}", w) for i, w in enumerate(Ws)], offs, "bf16")
        T = [C.cloak_tensor(o, n, k, C.CLOAK_BF16, C.CLOAK_ROWMAJOR) for (n, k), o in zip(shapes, offs)]
        X0 = {k: bf16_dev_from_bits(gen.synth(seed + 50, k, (batch, k), "bf16", kind=gen.KIND_NORMAL)) for k in {k for _, k in shapes}}
        n_ops = int(rng.integers(20, 61)) if small else int(rng.integers(1, 61))
        ops_c, ops_s, outs_c, outs_s, last_dep = [], [], [], [], False
        for j in range(n_ops):
            wi = int(rng.integers(0, n_w))
            n, k = shapes[wi]
            yc = torch.zeros(batch, n, dtype=torch.bfloat16, device="cuda")
            ys = torch.zeros_like(yc)
            # input: a fresh vector, or the output of an earlier op with matching width (a real dependency)
            cands = [i for i in range(j) if outs_c[i].shape[1] == k]
            if cands and rng.random() < 0.4:
                src = int(rng.choice(cands))
                xc, xs = outs_c[src], outs_s[src]
                after = 2 if (last_dep and rng.random() < 0.5) else 1
                last_dep = True
            else:
                xc = xs = X0[k]
                after = 0
            # gate epilogue from an earlier op of the same shape
            gates = [i for i in range(j) if ops_c[i][0] is T[wi]]
            if gates and rng.random() < 0.3:
                gi = int(rng.choice(gates))
                ac, as_ = torch.zeros_like(yc), torch.zeros_like(yc)
                ops_c.append((T[wi], xc, yc, after, outs_c[gi], ac))
                ops_s.append((T[wi], xs, ys, outs_s[gi], as_))
            else:
                ops_c.append((T[wi], xc, yc, after))
                ops_s.append((T[wi], xs, ys, None, None))
            outs_c.append(yc)
            outs_s.append(ys)
        # `after = 2` must follow a waiting op whose dependency covers it: make every dependent op wait for everything before it
        ops_c = [op if op[3] != 2 else op[:3] + (1,) + op[4:] for op in ops_c] if rng.random() < 0.5 else ops_c
        # an `after = 2` op shares the arrival of the nearest earlier waiting op, so its source must precede that op: enforce
        fixed, last_wait_at = [], -1
        for j, op in enumerate(ops_c):
            if op[3] == 1:
                last_wait_at = j
            if op[3] == 2:
                srcs = [i for i in range(j) if outs_c[i] is op[1]]
                if last_wait_at < 0 or (srcs and srcs[0] >= last_wait_at):
                    op = op[:3] + (1,) + op[4:]
                    last_wait_at = j
            fixed.append(op)
        C.cloak_gemv_chain(p.h, fixed, batch)
        for t, x, y, g, a_ in ops_s:
            C.cloak_gemv(p.h, t, x, y, batch)
            if g is not None:
                C.cloak_silu_mul(g, y, a_, y.numel(), C.CLOAK_BF16)
        torch.cuda.synchronize()
        for j in range(n_ops):
            assert torch.equal(outs_c[j], outs_s[j]), (seed, j, n_ops)
            if len(fixed[j]) == 6:
                assert torch.equal(fixed[j][5], ops_s[j][4]), (seed, j, "act")
        # against the oracle: every op whose input is a generator vector (never an oracle input from the CUDA path)
        Xh = {k: gen.synth(seed + 50, k, (batch, k), "bf16", kind=gen.KIND_NORMAL) for k in X0}
        for j in range(n_ops):
            if any(ops_s[j][1] is X0[k] for k in X0):
                wi = [i for i in range(n_w) if T[i] is ops_s[j][0]][0]
                check_linear(outs_c[j].float().cpu().numpy(), Xh[shapes[wi][1]], Ws[wi], "bf16", f"gemv_chain_random:s{seed}:op{j}", TOL["bf16"])


@pytest.mark.parametrize("seed", [0, 1, 2, 3, 4, 5])
def test_gemm_chain_random_lists(seed):
    """Random lists of 1..40 independent GEMMs (N, K from 128 to 3 584, any batch 1..256, random schedule: the static part, the
    dynamic chunk cap and therefore the number of contributors per tile row all vary; several launches past 16 ops): every
    op against the fp64 oracle, the whole list repeatable bit for bit and identical on the identity-table pool."""
    rng = np.random.default_rng(500 + seed)
    key, block, page = 0x1234, int(rng.choice([32768, 65536, 2 << 20])), 2 << 20
    batch = int(rng.choice([1, 5, 16, 24, 32, 77, 128, 256]))
    n_w = 5
    shapes = [(128 * int(rng.integers(1, 17)), 128 * int(rng.choice([1, 2, 3, 5, 8, 13, 28]))) for _ in range(n_w)]
    Ws = [gen.synth(seed, i, shp, "bf16") for i, shp in enumerate(shapes)]
    offs, total = C.cloak_arena_plan(key, [2 * n * k for n, k in shapes], block)
    sched = (int(rng.choice([0, 30, 75, 90, 100])), int(rng.choice([0, 1, 2, 5, 11, 40])))
    try:
        with Pool(total, block, page, key) as pc, Pool(total, block, page, key, C.CLOAK_POOL_IDENTITY) as pi:
            for (n, k), off, Wm in zip(shapes, offs, Ws):
                til = torch.empty(n * k, dtype=torch.bfloat16, device="cuda")
                C.cloak_to_tile128(bf16_dev_from_bits(Wm), til, n, k, C.CLOAK_BF16)
                for p in (pc, pi):
                    C.cloak_shuffle(p.h, til, off, n * k * 2)
            T = [C.cloak_tensor(o, n, k, C.CLOAK_BF16, C.CLOAK_TILE128) for (n, k), o in zip(shapes, offs)]
            X = {k: gen.synth(seed + 50, k, (batch, k), "bf16", kind=gen.KIND_NORMAL) for k in {k for _, k in shapes}}
            dX = {k: bf16_dev_from_bits(v) for k, v in X.items()}
            refs = [O.linear_f64(X[k], Wm) for (n, k), Wm in zip(shapes, Ws)]
            pick = [int(rng.integers(0, n_w)) for _ in range(int(rng.integers(1, 41)))]
            C.cloak_set_gemm_schedule(*sched)

            def run(pool):
                ys = [torch.zeros(batch, shapes[w][0], dtype=torch.bfloat16, device="cuda") for w in pick]
                C.cloak_gemm_chain(pool.h, [(T[w], dX[shapes[w][1]], y) for w, y in zip(pick, ys)], batch)
                torch.cuda.synchronize()
                return ys
            a, b, c = run(pc), run(pc), run(pi)
            for j, w in enumerate(pick):
                assert torch.equal(a[j], b[j]) and torch.equal(a[j], c[j]), (sched, batch, j, shapes[w])
                check_linear(a[j].float().cpu().numpy(), X[shapes[w][1]], Ws[w], "bf16",
                             f"gemm_chain_random:s{seed}:b{batch}:{sched[0]}/{sched[1]}:op{j}", TOL["bf16"])
    finally:
        C.cloak_set_gemm_schedule(75, 0)
