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
    ]
    for fn, st in cases:
        with pytest.raises(C.CloakError) as ei:
            fn()
        assert ei.value.status == st, C.cloak_last_error()
        assert C.cloak_last_error()


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
