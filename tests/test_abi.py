"""The C-ABI library loads, exports every symbol include/cloak.h declares, and rejects bad arguments
with the documented codes -- no GPU, no compute calls."""
import os
import re

import pytest

import oracle as O

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def C():
    import __graft_entry__
    __graft_entry__.build()
    import paper_2606_18400_b200 as C
    return C


def test_header_symbols_are_exported(C):
    hdr = open(os.path.join(ROOT, "include", "cloak.h")).read()
    declared = set(re.findall(r"\b(cloak_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(C.SYMBOLS), declared ^ set(C.SYMBOLS)
    for s in declared:
        assert getattr(C.lib, s) is not None
    assert "sm_100a" in C.cloak_version()


def test_arena_plan_matches_oracle_on_the_host(C):
    for key, sizes, b in [(0x1234, [x * 65536 for x in (512, 128, 128, 512, 1792, 1792, 1792)], 65536),
                          (0xFEED, [100, 4096, 1, 8191, 8192, 5000, 64, 12345], 4096),
                          (7, [16], 16), (0x1234, [2 * s[0] * s[1] for _, s in __import__("synth.gen", fromlist=["x"]).model_tensors(2)], 65536)]:
        offs, total = C.cloak_arena_plan(key, sizes, b)
        o_offs, o_total, _ = O.arena_plan(key, sizes, b)
        assert offs == o_offs and total == o_total


def test_argument_checks_without_a_device(C):
    cases = [
        (lambda: C.cloak_keygen(1, 2, 0, 16, 16), C.CLOAK_ERR_INVALID),
        (lambda: C.cloak_keygen(1, 2, 8, None, None), C.CLOAK_ERR_INVALID),
        (lambda: C.cloak_keygen(1, 2, (1 << 28) + 1, 16, 16), C.CLOAK_ERR_UNSUPPORTED),
        (lambda: C.cloak_pool_create(0, 0, 4096, 65536, 1), C.CLOAK_ERR_INVALID),
        (lambda: C.cloak_pool_create(0, 1 << 20, 3000, 65536, 1), C.CLOAK_ERR_UNSUPPORTED),
        (lambda: C.cloak_pool_create(0, 1 << 20, 4096, 65536 + 16, 1), C.CLOAK_ERR_ALIGN),
        (lambda: C.cloak_pool_create(0, 1 << 20, 4096, 65536, 1, 64), C.CLOAK_ERR_INVALID),
        (lambda: C.cloak_arena_plan(1, [], 4096), C.CLOAK_ERR_INVALID),
        (lambda: C.cloak_arena_plan(1, [10], 100), C.CLOAK_ERR_ALIGN),
        (lambda: C.cloak_set_copy_engine(9), C.CLOAK_ERR_INVALID),
        (lambda: C.cloak_to_tile128(16, 32, 100, 128, C.CLOAK_BF16), C.CLOAK_ERR_ALIGN),
        (lambda: C.cloak_silu_mul(None, None, None, 4, C.CLOAK_F32), C.CLOAK_ERR_INVALID),
        (lambda: C.cloak_relayout(None, None), C.CLOAK_ERR_INVALID),
        (lambda: C.cloak_pool_destroy(None), C.CLOAK_ERR_INVALID),
        # round 2's calls
        (lambda: C.cloak_pool_reserve_workspace(None, 1 << 20), C.CLOAK_ERR_INVALID),
        (lambda: C.cloak_rekey_pages_begin(None, 1, 1), C.CLOAK_ERR_INVALID),
        (lambda: C.cloak_rekey_pages_step(None, 1), C.CLOAK_ERR_INVALID),
        (lambda: C.cloak_rekey_pages_finish(None), C.CLOAK_ERR_INVALID),
        (lambda: C.cloak_pool_layout_report(None), C.CLOAK_ERR_INVALID),
        (lambda: C.cloak_pool_adjacency(None), C.CLOAK_ERR_INVALID),
        (lambda: C.cloak_pool_map_phases(None), C.CLOAK_ERR_INVALID),
        (lambda: C.cloak_set_copy_cache_hint(4), C.CLOAK_ERR_INVALID),
        (lambda: C.cloak_set_gather_engine(2), C.CLOAK_ERR_INVALID),
        (lambda: C.cloak_set_gemm_engine(4), C.CLOAK_ERR_INVALID),
        (lambda: C.cloak_set_gemv_engine(5), C.CLOAK_ERR_INVALID),
        (lambda: C.cloak_set_trace(12), C.CLOAK_ERR_ALIGN),
        (lambda: C.cloak_load_tensors(1, C.cloak_block_shape(256, 768, 4, 2, 64, C.CLOAK_BF16, 0), None, [(16, 0, 0, "gate")]), C.CLOAK_ERR_INVALID),
        (lambda: C.cloak_gemv_chain_scratch_bytes(None, [], 1), C.CLOAK_ERR_INVALID),
        (lambda: C.cloak_gemm_chain_scratch_bytes(None, [], 1), C.CLOAK_ERR_INVALID),
    ]
    for fn, st in cases:
        with pytest.raises(C.CloakError) as ei:
            fn()
        assert ei.value.status == st, C.cloak_last_error()
        assert C.cloak_last_error()


def test_runtime_info_and_knobs_are_callable_without_a_device(C):
    assert "gemv_chain" in C.cloak_runtime_info()
    C.cloak_set_copy_cache_hint(0)
    C.cloak_set_gather_engine(0)
    C.cloak_set_gemm_engine(0)
    C.cloak_set_trace(None)


def test_no_cpu_fallback(C):
    """Without a device the compute path must fail loudly, not fall back."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(C.CloakError) as ei:
        C.cloak_pool_create(0, 1 << 20, 4096, 65536, 1)
    assert ei.value.status == C.CLOAK_ERR_CUDA


def test_product_does_not_import_the_oracle():
    for base in ("paper_2606_18400_b200", "synth"):
        for dp, _, fs in os.walk(os.path.join(ROOT, base)):
            for f in fs:
                if f.endswith((".py", ".cu", ".cuh", ".h")):
                    txt = open(os.path.join(dp, f)).read()
                    assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, re.M), f
    for dp, _, fs in os.walk(os.path.join(ROOT, "oracle")):
        for f in fs:
            if f.endswith(".py"):
                txt = open(os.path.join(dp, f)).read()
                assert "paper_2606_18400_b200" not in re.sub(r'""".*?"""', "", txt, flags=re.S), f


def test_gemm_chunk_grid_on_the_host(C):
    """cloak_gemm_plan (the functions the tcgen05 GEMM kernel itself calls for its work split, run on the host): for the
    cfg1 / cfg3 layers and random op lists, under several schedules and row groupings -- the grouping is what cloak.h says
    (pairs by default only in launches of >= 160 tiles per SM whose matrices all have an even number of tile rows); the chunks
    cover the launch's unit sequence exactly once and in order; the static shares are equal to within one tile and there is one per CTA at most; every drawn chunk
    is non-empty and lies inside ONE tile row of ONE op (whole rows never split K); and a tile row is met by a bounded
    number of chunks (each extra one is a [batch x 128] fp32 partial and a share of a reduction)."""
    import numpy as np
    rng = np.random.default_rng(7)
    qwen = [(5120, 5120), (1024, 5120), (1024, 5120), (5120, 5120), (27648, 5120), (27648, 5120), (5120, 27648)]
    llama = [(4096, 4096), (1024, 4096), (1024, 4096), (4096, 4096), (14336, 4096), (14336, 4096), (4096, 14336)]
    lists = [qwen * 2, llama, qwen[:1], [(128, 128)], [(384, 640), (128, 128)]]
    lists += [[(128 * int(rng.integers(1, 40)), 128 * int(rng.integers(1, 60))) for _ in range(int(rng.integers(1, 17)))] for _ in range(20)]
    seen = set()
    try:
        for eng, sched in [(0, sc) for sc in ((75, 0), (100, 0), (0, 0), (40, 3), (90, 64))] + [(1, (75, 0)), (2, (75, 0)), (3, (75, 0)), (3, (0, 0))]:
            C.cloak_set_gemm_schedule(*sched)
            C.cloak_set_gemm_engine(eng)
            for shapes in lists:
                for batch, sms in ((1, 148), (32, 148), (128, 148), (256, 132), (77, 8), (64, 148)):
                    chunks, nstatic, g = C.cloak_gemm_plan(shapes, batch, sms)
                    mma = (batch + 15) // 16 * 16
                    # the grouping: a power of two that divides every matrix's tile rows, and whose accumulators (two buffers) fit TMEM
                    assert g in (1, 2, 4) and all((n // 128) % g == 0 for n, _ in shapes) and 2 * g * mma <= 512, (eng, shapes, batch, g)
                    if eng == 1 or (eng == 0 and (mma < 32 or sum((n // 128) * (k // 128) for n, k in shapes) < 160 * sms)):
                        assert g == 1
                    if eng == 3 and mma <= 128 and all((n // 128) % 2 == 0 for n, _ in shapes):
                        assert g == 2
                    if eng == 2 and mma <= 64 and all((n // 128) % 4 == 0 for n, _ in shapes):
                        assert g == 4
                    seen.add((eng, g))
                    total = sum((n // 128 // g) * (k // 128) for n, k in shapes)
                    assert 1 <= nstatic <= sms
                    # group-row boundaries of the sequence: op j, group row r starts at ubase_j + r * kt_j
                    starts, kts, u = [], [], 0
                    for n, k in shapes:
                        for r in range(n // 128 // g):
                            starts.append(u + r * (k // 128))
                            kts.append(k // 128)
                        u += (n // 128 // g) * (k // 128)
                    starts = np.array(starts)
                    pos = 0
                    sizes = []
                    for c, (b, e) in enumerate(chunks):
                        assert b == pos and e >= b, (sched, shapes, batch, c)
                        pos = e
                        if c < nstatic:
                            sizes.append(e - b)
                        else:
                            assert e > b
                            r = int(np.searchsorted(starts, b, side="right")) - 1
                            assert e <= starts[r] + kts[r], (sched, shapes, batch, c)       # inside one group row
                    assert pos == total
                    assert max(sizes) - min(sizes) <= 1
                    # chunks per group row
                    edges = np.array([b for b, e in chunks if e > b])
                    first = np.searchsorted(edges, starts, side="right") - 1
                    last = np.searchsorted(edges, starts + np.array(kts) - 1, side="right") - 1
                    per_row = last - first + 1
                    if sched[1] == 0:
                        assert per_row.max() <= 12, (sched, shapes, batch, int(per_row.max()))
        assert {(0, 1), (0, 2), (1, 1), (2, 4), (2, 2), (3, 2), (3, 1)} <= seen, seen
    finally:
        C.cloak_set_gemm_schedule(75, 0)
        C.cloak_set_gemm_engine(0)
    for bad in [([(100, 128)], 32, 148), ([(128, 128)] * 17, 32, 148), ([(128, 128)], 0, 148), ([(128, 128)], 32, 0)]:
        with pytest.raises(C.CloakError):
            C.cloak_gemm_plan(*bad)
