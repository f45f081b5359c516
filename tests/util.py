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
