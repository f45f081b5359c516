"""O9, O11, O12 -- the contraction the authorised read must reach, in fp64.  Test oracle.

Paper: the authorised reader keeps "a valid logical memory view" and runs at
"near-native performance" because "LLM inference is bandwidth-bound".
BJ:north_star (c): "a permutation-aware decode GEMV/GEMM that gathers weight tiles through the
block-permutation table"; tolerance "max relative error <= 2e-2 for bf16 and <= 1e-5 for fp32
accumulators on fp32 inputs" against an fp32 oracle.

O11: Y[m, n] = sum_k X[m, k] * W[n, k]; inputs converted exactly to fp64, summed in fp64, emitted
as fp32 (G17).  W is the *logical* matrix: the oracle never touches a shuffled layout here.
bf16 values travel as uint16 bit patterns (numpy has no bf16).
"""
import numpy as np


def bf16_bits_to_f32(u16):
    u = np.asarray(u16, dtype=np.uint16).astype(np.uint32) << np.uint32(16)
    return u.view(np.float32)


def f32_to_bf16_bits(x):
    """Round-to-nearest-even fp32 -> bf16 bit pattern (finite inputs)."""
    u = np.asarray(x, dtype=np.float32).view(np.uint32).astype(np.uint64)
    lsb = (u >> np.uint64(16)) & np.uint64(1)
    u = u + np.uint64(0x7FFF) + lsb
    return (u >> np.uint64(16)).astype(np.uint16)


def to_f64(a):
    """Exact conversion of an fp32 array, or a uint16 array of bf16 bits, to fp64."""
    a = np.asarray(a)
    if a.dtype == np.uint16:
        return bf16_bits_to_f32(a).astype(np.float64)
    if a.dtype in (np.float32, np.float64):
        return a.astype(np.float64)
    raise TypeError("expected float32 or uint16 (bf16 bits)")


def linear_f64(X, W):
    """O11.  X [batch, K], W [N, K] (fp32 or bf16 bits) -> Y [batch, N] float32."""
    return (to_f64(X) @ to_f64(W).T).astype(np.float32)


def silu(z):
    return z / (1.0 + np.exp(-z))


def mlp_f64(x, gate, up, down):
    """O9: MLP(x) = down . (silu(gate . x) * (up . x)), all fp64.  x [batch, H] -> [batch, H] fp64."""
    x = to_f64(x)
    g = x @ to_f64(gate).T
    u = x @ to_f64(up).T
    return (silu(g) * u) @ to_f64(down).T


def attention_f64(x, q, k, v, o, n_q, n_kv, d):
    """Brute-force causal softmax attention with grouped KV heads, fp64 (O9).

    x [tokens, H]; q [n_q*d, H]; k, v [n_kv*d, H]; o [H, n_q*d].  Query head h uses KV head h // G.
    No rotary embedding and no norms (G15): those act inside a head, which O8 never reorders.
    """
    x = to_f64(x)
    t = x.shape[0]
    G = n_q // n_kv
    Q = (x @ to_f64(q).T).reshape(t, n_q, d)
    K = (x @ to_f64(k).T).reshape(t, n_kv, d)
    V = (x @ to_f64(v).T).reshape(t, n_kv, d)
    ctx = np.zeros((t, n_q, d), dtype=np.float64)
    for h in range(n_q):
        g = h // G
        for i in range(t):
            s = np.array([Q[i, h] @ K[j, g] for j in range(i + 1)]) / np.sqrt(d)
            p = np.exp(s - s.max())
            p /= p.sum()
            for j in range(i + 1):
                ctx[i, h] += p[j] * V[j, g]
    return ctx.reshape(t, n_q * d) @ to_f64(o).T


def to_tile128(W):
    """O11 CLOAK_TILE128 storage of a logical [N, K] matrix (N, K multiples of 128).

    Tile (tn, tk) sits at tile index tn*(K/128) + tk; element (r, c) of the tile at element offset
    r*128 + c inside it; plain row-major inside the tile, no swizzle.  Returns a flat array.
    """
    N, K = W.shape
    if N % 128 or K % 128:
        raise ValueError("TILE128 needs N and K multiples of 128")
    return W.reshape(N // 128, 128, K // 128, 128).transpose(0, 2, 1, 3).copy().ravel()


def from_tile128(flat, N, K):
    return flat.reshape(N // 128, K // 128, 128, 128).transpose(0, 2, 1, 3).copy().reshape(N, K)


def err_normwise(y, y_ref):
    """O12 gated number: max_i |y_i - yref_i| / max_i |yref_i|."""
    y = np.asarray(y, dtype=np.float64)
    y_ref = np.asarray(y_ref, dtype=np.float64)
    return float(np.max(np.abs(y - y_ref)) / np.max(np.abs(y_ref)))


def err_elementwise_floored(y, y_ref):
    """O12 reported number: max_i |y_i - yref_i| / max(|yref_i|, rms(yref))."""
    y = np.asarray(y, dtype=np.float64)
    y_ref = np.asarray(y_ref, dtype=np.float64)
    rms = np.sqrt(np.mean(y_ref ** 2))
    return float(np.max(np.abs(y - y_ref) / np.maximum(np.abs(y_ref), rms)))
