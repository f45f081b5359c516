"""Writes tests/golden/moe_example.json: worked values of the MoE permutation streams ("MoE layers").

Independent of oracle/ and of the CUDA path on purpose: Philox4x32-10 is restated here from its round function in plain
Python integers (constants 0xD2511F53, 0xCD9E8D57, key bumps 0x9E3779B9, 0xBB67AE85, ten rounds), the sort key is
r_i = o0:o1 of counter (i, 0, stream lo, stream hi), and a permutation is `sorted(range(n), key=(r_i, i))` (O2).  The streams
are EXPERT = (7<<32)|layer and EXPERT_MLP = (8<<32)|(layer*E + e).  tests/test_oracle_pins.py checks that the numpy oracle
reproduces every value stored here.

    python tests/golden/make_moe_example.py
"""
import json
import os

M32 = 0xFFFFFFFF


def philox(ctr, key):
    c0, c1, c2, c3 = ctr
    k0, k1 = key
    for _ in range(10):
        p0, p1 = 0xD2511F53 * c0, 0xCD9E8D57 * c2
        c0, c1, c2, c3 = ((p1 >> 32) ^ c1 ^ k0) & M32, p1 & M32, ((p0 >> 32) ^ c3 ^ k1) & M32, p0 & M32
        k0, k1 = (k0 + 0x9E3779B9) & M32, (k1 + 0xBB67AE85) & M32
    return c0, c1, c2, c3


def perm(key, stream, n):
    r = []
    for i in range(n):
        o = philox((i & M32, i >> 32, stream & M32, stream >> 32), (key & M32, key >> 32))
        r.append((o[0] << 32) | o[1])
    return sorted(range(n), key=lambda i: (r[i], i))


def fnv(a):
    h = 0xCBF29CE484222325
    for v in a:
        for b in int(v).to_bytes(4, "little"):
            h = ((h ^ b) * 0x100000001B3) & 0xFFFFFFFFFFFFFFFF
    return f"{h:016x}"


if __name__ == "__main__":
    # self-check against SURVEY.md 8(c).3's worked examples before anything is written
    assert perm(0x1234, 0, 16) == [1, 7, 11, 8, 5, 0, 9, 13, 15, 10, 2, 14, 12, 3, 6, 4]
    assert perm(0x1234, 1 << 32, 16) == [8, 4, 14, 1, 2, 11, 10, 7, 12, 15, 9, 0, 6, 5, 3, 13]
    key, out = 0x1234, {"_citation": __doc__.split("\n")[0] + "  Made by tests/golden/make_moe_example.py (pure-Python restatement, "
                        "independent of oracle/).", "key": "0x1234", "cases": []}
    for layer, E, I, experts in ((3, 6, 12, (0, 5)), (0, 128, 768, (0, 77, 127)), (47, 128, 768, (5,))):
        eps = perm(key, (7 << 32) | layer, E)
        case = {"layer": layer, "n_experts": E, "inter": I, "eps_head": eps[:8], "fnv_eps": fnv(eps), "pi": []}
        if E <= 8:
            case["eps"] = eps
        for e in experts:
            pi = perm(key, (8 << 32) | (layer * E + e), I)
            case["pi"].append({"expert": e, "head": pi[:8], "fnv": fnv(pi), **({"perm": pi} if I <= 16 else {})})
        out["cases"].append(case)
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "moe_example.json")
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
        f.write("\n")
    print("wrote", path)
