"""Re-derive the bit patterns stored in tests/golden/*.json from exact rationals.

Calls neither the CUDA library nor the oracle: squared distances are exact Fractions of the
dyadic coordinates, distances are their square roots to 60 decimal digits rounded to the nearest
binary32, clearances one binary32 subtraction (numpy).  Run: ``python tests/golden/check_golden.py``.
"""
import glob
import json
import os
import struct
from decimal import Decimal, getcontext
from fractions import Fraction

import numpy as np

getcontext().prec = 60


def f32_bits_of(x: Decimal) -> int:
    b = struct.unpack("<I", struct.pack("<f", float(x)))[0]
    cands = [bb for bb in (b - 1, b, b + 1) if 0 <= bb < 0x7F800000]
    return min(cands, key=lambda bb: abs(Decimal(struct.unpack("<f", struct.pack("<I", bb))[0]) - x))


def bits(f) -> str:
    return "%08x" % struct.unpack("<I", struct.pack("<f", float(f)))[0]


def check_scene(path):
    g = json.load(open(path))
    P = [[Fraction(v) for v in row] for row in g["points"]]
    n = len(P)
    for i in range(n):
        keys = sorted((sum((a - b) ** 2 for a, b in zip(P[i], P[j])), j) for j in range(n) if j != i)
        (s1, j1), (s2, j2) = keys[0], keys[1]
        assert j1 == g["nn"][i] and j2 == g["nn2"][i], (path, i)
        assert s1 == Fraction(g["s1"][i]) and s2 == Fraction(g["s2"][i]), (path, i)
        d1 = f32_bits_of((Decimal(s1.numerator) / Decimal(s1.denominator)).sqrt())
        d2 = f32_bits_of((Decimal(s2.numerator) / Decimal(s2.denominator)).sqrt())
        if "d1_bits" in g:
            assert "%08x" % d1 == g["d1_bits"][i] and "%08x" % d2 == g["d2_bits"][i], (path, i)
        f1 = np.float32(struct.unpack("<f", struct.pack("<I", d1))[0])
        f2 = np.float32(struct.unpack("<f", struct.pack("<I", d2))[0])
        assert bits(f2 - f1) == g["c_bits"][i], (path, i)


def check_topk(path):
    """K-list certificates (reading R20): lists, exact squared distances, distance and clearance bits."""
    for g in json.load(open(path))["scenes"]:
        P = [[Fraction(v) for v in row] for row in g["points"]]
        n, K = len(P), g["K"]
        for i in range(n):
            keys = sorted((sum((a - b) ** 2 for a, b in zip(P[i], P[j])), j) for j in range(n) if j != i)[:K]
            assert [j for _, j in keys] == g["nnk"][i], (path, i)
            assert [s for s, _ in keys] == [Fraction(v) for v in g["sk"][i]], (path, i)
            db = [f32_bits_of((Decimal(s.numerator) / Decimal(s.denominator)).sqrt()) for s, _ in keys]
            assert ["%08x" % b for b in db] == g["dk_bits"][i], (path, i)
            f = [np.float32(struct.unpack("<f", struct.pack("<I", b))[0]) for b in db]
            assert bits(f[K - 1] - f[K - 2]) == g["ck_bits"][i], (path, i)


if __name__ == "__main__":
    here = os.path.dirname(os.path.abspath(__file__))
    for f in sorted(glob.glob(os.path.join(here, "p[12]*.json"))):
        check_scene(f)
        print("ok", os.path.basename(f))
    check_topk(os.path.join(here, "p7_topk_lists.json"))
    print("ok p7_topk_lists.json")
