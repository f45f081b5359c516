"""Seeded synthetic inputs shared by the oracle side and the CUDA side (numpy twin).

This module is the *input generator* only: it holds none of the method's arithmetic (no Philox,
no tables, no layout).  Both `tests/` and `bench.py` draw weights and activations from it; its
CUDA twin (`synth/csrc/synth_fill.cu`, built as `synth/libcloaksynth.so`) fills device buffers
with byte-identical values so multi-GB configs never cross PCIe.  A GPU test checks the twins
agree byte for byte.

The values stand in for the paper's Llama 3.1 8B / Qwen3 checkpoints, which are not in the
container: only the *shapes* come from those models ("weights ~N(0,0.02)", BJ:configs).

Generator (element x of tensor t under seed s; all arithmetic mod 2^64):
    mix(z):  z ^= z >> 30;  z *= 0xBF58476D1CE4E5B9;  z ^= z >> 27;  z *= 0x94D049BB133111EB;
             z ^= z >> 31                                   (the splitmix64 output function)
    base = mix( mix(s + GOLD) ^ (t * 0xD1B54A32D192ED03 + 0x8CB92BA72F3D8DD7) )
    h1 = mix(base + (2x) * GOLD),  h2 = mix(base + (2x + 1) * GOLD),  GOLD = 0x9E3779B97F4A7C15
    S  = sum of the eight 16-bit fields of h1 and h2        (Irwin-Hall, 8 terms)
    z  = S - 262140 (integer);   w = fp32(z) * c            (one fp32 multiply)
    c  = 0x34C8A986 (= 0.02 / sigma_S) for weights, 0x379CC471 (= 1 / sigma_S) for N(0,1) inputs,
         sigma_S = sqrt(8 * (65536^2 - 1) / 12) = 53509.92
    bf16 configs: round-to-nearest-even of w to bf16.
Excess kurtosis -0.15, support +-4.9 sigma.  "~N(0,0.02)" is read as sigma = 0.02 (O10).
This replaces SURVEY.md O10's Philox-based recipe so that the shared module carries no Philox;
worked example W6 therefore does not apply (recorded in DESIGN.md, readings).
"""
import numpy as np

GOLD = np.uint64(0x9E3779B97F4A7C15)
_C1 = np.uint64(0xBF58476D1CE4E5B9)
_C2 = np.uint64(0x94D049BB133111EB)
_T1 = np.uint64(0xD1B54A32D192ED03)
_T2 = np.uint64(0x8CB92BA72F3D8DD7)
SCALE_WEIGHT = np.array([0x34C8A986], dtype=np.uint32).view(np.float32)[0]
SCALE_NORMAL = np.array([0x379CC471], dtype=np.uint32).view(np.float32)[0]
KIND_WEIGHT, KIND_NORMAL = 0, 1


def _mix(z):
    z = z ^ (z >> np.uint64(30))
    z = z * _C1
    z = z ^ (z >> np.uint64(27))
    z = z * _C2
    return z ^ (z >> np.uint64(31))


def _sum16(h):
    m = np.uint64(0xFFFF)
    return ((h & m) + ((h >> np.uint64(16)) & m) + ((h >> np.uint64(32)) & m)
            + (h >> np.uint64(48))).astype(np.int64)


def synth_f32(seed, tensor, start, count, kind=KIND_WEIGHT):
    """fp32 values of elements [start, start+count) of tensor `tensor` under `seed`."""
    with np.errstate(over="ignore"):
        s = np.array([seed], dtype=np.uint64)
        t = np.array([tensor], dtype=np.uint64)
        base = _mix(_mix(s + GOLD) ^ (t * _T1 + _T2))
        x = np.arange(start, start + count, dtype=np.uint64)
        h1 = _mix(base + (x * np.uint64(2)) * GOLD)
        h2 = _mix(base + (x * np.uint64(2) + np.uint64(1)) * GOLD)
    z = _sum16(h1) + _sum16(h2) - 262140
    c = SCALE_WEIGHT if kind == KIND_WEIGHT else SCALE_NORMAL
    return z.astype(np.float32) * c


def f32_to_bf16_bits(x):
    u = np.asarray(x, dtype=np.float32).view(np.uint32).astype(np.uint64)
    u = u + np.uint64(0x7FFF) + ((u >> np.uint64(16)) & np.uint64(1))
    return (u >> np.uint64(16)).astype(np.uint16)


def synth_bf16_bits(seed, tensor, start, count, kind=KIND_WEIGHT):
    return f32_to_bf16_bits(synth_f32(seed, tensor, start, count, kind))


def synth(seed, tensor, shape, dtype, kind=KIND_WEIGHT, start=0):
    """Whole tensor: dtype 'f32' -> float32 array, 'bf16' -> uint16 bit patterns."""
    n = int(np.prod(shape))
    out = np.empty(n, dtype=np.float32 if dtype == "f32" else np.uint16)
    step = 1 << 22
    for a in range(0, n, step):
        c = min(step, n - a)
        v = synth_f32(seed, tensor, start + a, c, kind)
        out[a:a + c] = v if dtype == "f32" else f32_to_bf16_bits(v)
    return out.reshape(shape)


# Model shapes of BJ:configs (Linear convention [out, in]); canonical order q,k,v,o,gate,up,down (O7).
def layer_shapes(hidden, inter, n_q, n_kv, head_dim):
    return [("q", (n_q * head_dim, hidden)), ("k", (n_kv * head_dim, hidden)),
            ("v", (n_kv * head_dim, hidden)), ("o", (hidden, n_q * head_dim)),
            ("gate", (inter, hidden)), ("up", (inter, hidden)), ("down", (hidden, inter))]


CONFIGS = {
    # cfg0: tiny fp32 MLP block (BJ:configs[0])
    0: dict(seed=0, key=0x1234, dtype="f32", hidden=256, inter=1024, block=4096, page=65536),
    # cfg1: one LLaMA-8B-shaped decoder layer (BJ:configs[1])
    1: dict(seed=1, key=0x1234, dtype="bf16", hidden=4096, inter=14336, n_q=32, n_kv=8, head_dim=128,
            block=65536, page=2 << 20, layers=1),
    # cfg2: full 32-layer LLaMA-8B shape (BJ:configs[2]); tensors = embed, 32 x 7, lm_head (G10)
    2: dict(seed=2, key=0x1234, dtype="bf16", hidden=4096, inter=14336, n_q=32, n_kv=8, head_dim=128,
            block=65536, page=2 << 20, layers=32, vocab=128256),
    # cfg3: Qwen-32B shape, layers only (BJ:configs[3], G9)
    3: dict(seed=3, key=0x1234, dtype="bf16", hidden=5120, inter=27648, n_q=40, n_kv=8, head_dim=128,
            block=65536, page=2 << 20, layers=64),
    # cfg4: 4 GiB granularity sweep (BJ:configs[4]); key B = 0x5678 (G11)
    4: dict(seed=4, key=0x1234, key_b=0x5678, dtype="bf16", bytes=4 << 30, page=2 << 20,
            blocks=[4 << 10, 16 << 10, 64 << 10, 256 << 10, 2 << 20]),
    # cfg5 (NEXT-4, not in BASELINE.json): Qwen3-30B-A3B-shaped sparse layers (the paper's MoE model)
    5: dict(seed=5, key=0x1234, dtype="bf16", hidden=2048, inter=768, n_experts=128, top_k=8, n_q=32, n_kv=4, head_dim=128,
            block=65536, page=2 << 20, layers=48),
}


def model_tensors(cfg):
    """Canonical tensor list [(name, shape)] of a model config (O7 order)."""
    c = CONFIGS[cfg]
    out = []
    if "vocab" in c:
        out.append(("embed", (c["vocab"], c["hidden"])))
    for l in range(c.get("layers", 1)):
        for nm, shp in layer_shapes(c["hidden"], c["inter"], c["n_q"], c["n_kv"], c["head_dim"]):
            out.append((f"l{l}.{nm}", shp))
    if "vocab" in c:
        out.append(("lm_head", (c["vocab"], c["hidden"])))
    return out
