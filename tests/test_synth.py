"""The shared seeded input generator (synth/gen.py): determinism and distribution.  CPU-only."""
import numpy as np
from synth import gen


def test_chunking_and_determinism():
    a = gen.synth_f32(1, 6, 0, 10000)
    b = np.concatenate([gen.synth_f32(1, 6, 0, 3333), gen.synth_f32(1, 6, 3333, 6667)])
    assert np.array_equal(a, b)
    assert not np.array_equal(a, gen.synth_f32(2, 6, 0, 10000))
    assert not np.array_equal(a, gen.synth_f32(1, 5, 0, 10000))
    # python-int restatement of the recipe for a few elements
    M = (1 << 64) - 1

    def mix(z):
        z ^= z >> 30
        z = (z * 0xBF58476D1CE4E5B9) & M
        z ^= z >> 27
        z = (z * 0x94D049BB133111EB) & M
        return z ^ (z >> 31)

    G = 0x9E3779B97F4A7C15
    base = mix(mix((1 + G) & M) ^ ((6 * 0xD1B54A32D192ED03 + 0x8CB92BA72F3D8DD7) & M))
    for x in (0, 1, 77, 9999):
        S = 0
        for h in (mix((base + 2 * x * G) & M), mix((base + (2 * x + 1) * G) & M)):
            S += sum((h >> s) & 0xFFFF for s in (0, 16, 32, 48))
        assert a[x] == np.float32(S - 262140) * gen.SCALE_WEIGHT


def test_distribution():
    w = gen.synth_f32(0, 0, 0, 1 << 22).astype(np.float64)
    assert abs(w.mean()) < 1e-4
    assert abs(w.std() - 0.02) < 0.02 * 0.01
    assert np.abs(w).max() < 4.9 * 0.02
    x = gen.synth_f32(0, 1, 0, 1 << 20, gen.KIND_NORMAL).astype(np.float64)
    assert abs(x.std() - 1.0) < 0.01
    # element index beyond 2^32 works (cfg2/3/4 offsets)
    assert gen.synth_f32(4, 0, (1 << 33) + 5, 4).shape == (4,)


def test_model_tensor_lists():
    assert len(gen.model_tensors(1)) == 7
    t2 = gen.model_tensors(2)
    assert len(t2) == 226 and t2[0][0] == "embed" and t2[-1][0] == "lm_head"
    assert sum(2 * s[0] * s[1] for _, s in t2) == 16059990016
    t3 = gen.model_tensors(3)
    assert len(t3) == 448 and sum(2 * s[0] * s[1] for _, s in t3) == 62411243520
    assert sum(2 * s[0] * s[1] for _, s in gen.model_tensors(1)) == 436207616
