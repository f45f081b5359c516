"""cloak_gemv_static: the cloaked GEMV with its scratch in the library's fixed `static __device__` array -- the entry point
that allocates nothing (cloak.h).  Checked against the existing path (cloak_gemv, scratch in the pool's workspace): the same
kernel on the same split, so bit for bit, and against the oracle within the tolerance every GEMV test uses.

This file is collected LAST on purpose (the suite runs with `pytest -x`); it passes alone in a fresh process and after the
other tests -- the static array keeps whatever an earlier call left in it, which is what the back-to-back calls exercise.
"""
import pytest
import torch

from synth import gen
from util import check_linear

pytestmark = pytest.mark.gpu

if torch.cuda.is_available():
    import paper_2606_18400_b200 as C
    from gpu_util import Pool, bf16_dev_from_bits

TOL = 2e-2                          # bf16, O12 norm-wise (BASELINE.json north_star); check_linear adds the arithmetic bound
SHAPES = [(4096, 14336), (1024, 4096), (48, 1024), (5120, 5120)]      # cut row tiles (kch > 1), one chunk per row, ragged N / 16, 2.5 KiB chunks


def _setup(key=0x1234, seed=21, block=65536, page=2 << 20):
    Ws = [gen.synth(seed, i, shp, "bf16") for i, shp in enumerate(SHAPES)]
    offs, total = C.cloak_arena_plan(key, [2 * n * k for n, k in SHAPES], block)
    pool = Pool(total, block, page, key)
    for Wm, off in zip(Ws, offs):
        d = bf16_dev_from_bits(Wm)
        C.cloak_shuffle(pool.h, d, off, d.numel() * 2)
    T = [C.cloak_tensor(o, n, k, C.CLOAK_BF16, C.CLOAK_ROWMAJOR) for (n, k), o in zip(SHAPES, offs)]
    return pool, Ws, T


def test_gemv_static_equals_the_workspace_path_on_calls_in_a_row():
    pool, Ws, T = _setup()
    try:
        seq = [(0, 1), (0, 16), (1, 4), (2, 8), (3, 16), (0, 3), (3, 1), (0, 1)]      # (tensor, batch): big after small, small after big, repeats
        X = {(w, b): gen.synth(121, 16 * w + b, (b, SHAPES[w][1]), "bf16", kind=gen.KIND_NORMAL) for w, b in seq}
        dX = {k: bf16_dev_from_bits(v) for k, v in X.items()}
        ref = [torch.zeros(b, SHAPES[w][0], dtype=torch.bfloat16, device="cuda") for w, b in seq]
        got = [torch.full((b, SHAPES[w][0]), 7.0, dtype=torch.bfloat16, device="cuda") for w, b in seq]
        for (w, b), y in zip(seq, ref):                       # the existing path
            C.cloak_gemv(pool.h, T[w], dX[w, b], y, b)
        warm = torch.zeros(1, SHAPES[2][0], dtype=torch.bfloat16, device="cuda")
        C.cloak_gemv_static(pool.h, T[2], dX[2, 8], warm, 1)  # set-up: the symbol's address on this device, the kernels' code resident
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        launches0 = C.cloak_launch_count()
        for (w, b), y in zip(seq, got):                       # the new entry point: all calls in a row, nothing in between
            C.cloak_gemv_static(pool.h, T[w], dX[w, b], y, b)
        torch.cuda.synchronize()
        assert C.cloak_launch_count() - launches0 == 2 * len(seq)
        assert torch.cuda.mem_get_info()[0] >= free0          # nothing was allocated on the device
        for i, ((w, b), y, r) in enumerate(zip(seq, got, ref)):
            assert torch.equal(y, r), (i, w, b)
            if i < 5:
                check_linear(y.float().cpu().numpy(), X[w, b], Ws[w], "bf16", f"gemv_static:{SHAPES[w][0]}x{SHAPES[w][1]}:b{b}", TOL)
        # on a side stream, and captured into a CUDA graph (capture forbids cudaMalloc: the call must not need it)
        side = torch.cuda.Stream()
        y2 = torch.zeros_like(ref[1])
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            C.cloak_gemv_static(pool.h, T[0], dX[0, 16], y2, 16, stream=side)
        side.synchronize()
        assert torch.equal(y2, ref[1])
        y3, y4 = torch.zeros_like(ref[1]), torch.zeros_like(ref[2])
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            C.cloak_gemv_static(pool.h, T[0], dX[0, 16], y3, 16)
            C.cloak_gemv_static(pool.h, T[1], dX[1, 4], y4, 4)
        for _ in range(2):
            y3.zero_()
            y4.zero_()
            g.replay()
            torch.cuda.synchronize()
            assert torch.equal(y3, ref[1]) and torch.equal(y4, ref[2])
    finally:
        torch.cuda.synchronize()
        pool.close()


def test_gemv_static_rejects_what_the_fixed_scratch_cannot_hold():
    big_n = 524288 + 16                                       # one row-tile counter per 8 rows: 65 536 counters hold N <= 524 288
    pool = Pool(2 * big_n * 256, 65536, 2 << 20, 0x1234)
    try:
        x = torch.zeros(16, 256, dtype=torch.bfloat16, device="cuda")
        y = torch.zeros(16, big_n, dtype=torch.bfloat16, device="cuda")
        launches0 = C.cloak_launch_count()
        cases = [(C.cloak_tensor(0, big_n, 256, C.CLOAK_BF16, C.CLOAK_ROWMAJOR), 1, C.CLOAK_ERR_UNSUPPORTED, "static scratch"),
                 (C.cloak_tensor(0, 1024, 256, C.CLOAK_F32, C.CLOAK_ROWMAJOR), 1, C.CLOAK_ERR_UNSUPPORTED, "CLOAK_BF16"),
                 (C.cloak_tensor(0, 1024, 320, C.CLOAK_BF16, C.CLOAK_ROWMAJOR), 1, C.CLOAK_ERR_UNSUPPORTED, "K % 256"),
                 (C.cloak_tensor(0, 1024, 256, C.CLOAK_BF16, C.CLOAK_TILE128), 1, C.CLOAK_ERR_UNSUPPORTED, "ROWMAJOR"),
                 (C.cloak_tensor(0, 1024, 256, C.CLOAK_BF16, C.CLOAK_ROWMAJOR), 17, C.CLOAK_ERR_INVALID, "batch")]
        for t, b, status, word in cases:
            with pytest.raises(C.CloakError) as ei:
                C.cloak_gemv_static(pool.h, t, x, y, b)
            assert ei.value.status == status and word in C.cloak_last_error(), C.cloak_last_error()
        assert C.cloak_launch_count() == launches0            # nothing was launched
        # the largest N it takes: runs, and equals the workspace path
        t = C.cloak_tensor(0, 524288, 256, C.CLOAK_BF16, C.CLOAK_ROWMAJOR)
        x.copy_(torch.randn(16, 256, device="cuda").bfloat16())
        w = torch.randn(524288 * 256 // 64, 64, device="cuda").bfloat16()
        C.cloak_shuffle(pool.h, w, 0, w.numel() * 2)
        y1, y2 = torch.zeros(2, 524288, dtype=torch.bfloat16, device="cuda"), torch.zeros(2, 524288, dtype=torch.bfloat16, device="cuda")
        C.cloak_gemv(pool.h, t, x, y1, 2)
        C.cloak_gemv_static(pool.h, t, x, y2, 2)
        torch.cuda.synchronize()
        assert torch.equal(y1, y2) and float(y1.float().abs().sum()) > 0
    finally:
        torch.cuda.synchronize()
        pool.close()
