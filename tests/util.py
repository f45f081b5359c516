"""Small helpers shared by the tests (no method arithmetic)."""
import json
import os
import numpy as np

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def fnv1a64_u32(a):
    """FNV-1a-64 over the little-endian uint32 array (checksum used by SURVEY.md 8(c).3)."""
    h = 0xCBF29CE484222325
    for byte in np.asarray(a, dtype="<u4").tobytes():
        h = ((h ^ byte) * 0x100000001B3) & 0xFFFFFFFFFFFFFFFF
    return f"{h:016x}"


def worked():
    with open(os.path.join(GOLDEN, "worked_examples.json")) as f:
        return json.load(f)


def philox_kat():
    rows = []
    with open(os.path.join(GOLDEN, "philox_kat.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            w = line.split()
            rows.append(([int(x, 16) for x in w[:6]], [None if x == "-" else int(x, 16) for x in w[6:]]))
    return rows


# ---- O12 error report + the tight gate derived from the arithmetic ("tolerances")
ERRLOG = []        # (tag, dtype, err_normwise, err_elementwise_floored, worst |diff| / bound); conftest prints it at the end


def check_linear(got, X, W, dtype, tag, tol):
    """One GEMV / GEMM output `got` [batch, N] (float array) against the oracle's O11 contraction of X [batch, K], W [N, K].

    Two gates.  (1) The contract's: O12 norm-wise error <= tol (2e-2 bf16, 1e-5 fp32; BASELINE.json north_star).
    (2) A bound that follows from the arithmetic alone, element by element.  Both sides start from the same bf16 / fp32
    inputs; a product of two bf16 values is exact in fp32; the kernel sums K products in fp32 in SOME order (warp slices,
    split-K partials, MMA accumulators: each addition rounds or truncates, |error| <= 2^-23 of the partial sum), and rounds
    the result once to the output type (bf16: relative 2^-8; fp32: nothing further, but its products round too: 2^-24
    each).  Hence, with A_i = sum_k |x_k| |w_ik| computed by the oracle in fp64,
        |y_i - yref_i|  <=  r * |yref_i|  +  (1 + r) * K * 2^-23 * A_i,      r = 2^-8 (bf16 out) or 2^-24 (fp32 out),
    for any summation order.  A dropped 64-byte k-step (32 of K = 4096 terms) moves y_i by ~0.09 rms(y), five times what
    this allows at |y_i| ~ rms(y), while it would pass the norm-wise 2e-2.  Both errors and the worst ratio are logged.
    """
    import oracle as O
    got = np.asarray(got, dtype=np.float64)
    ref = O.linear_f64(X, W).astype(np.float64)
    A = np.abs(O.to_f64(X)) @ np.abs(O.to_f64(W)).T
    K = np.asarray(X).shape[-1]
    r = 2.0 ** -8 if dtype == "bf16" else 2.0 ** -24
    bound = r * np.abs(ref) + (1 + r) * K * 2.0 ** -23 * A + 1e-30
    en, ee = O.err_normwise(got, ref), O.err_elementwise_floored(got, ref)
    worst = float(np.max(np.abs(got - ref) / bound))
    ERRLOG.append((tag, dtype, en, ee, worst))
    assert en <= tol, (tag, "O12 norm-wise", en)
    assert worst <= 1.0, (tag, "arithmetic bound exceeded", worst, en, ee)
    return en, ee
