"""Reader of the `key = value` fixtures under tests/golden/ (values may be decimals or exact rationals p/q)."""
import os
from fractions import Fraction

HERE = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def load(name):
    out = {}
    for line in open(os.path.join(HERE, name)):
        line = line.split("#", 1)[0].strip()
        if not line:
            continue
        k, v = [x.strip() for x in line.split("=", 1)]
        out[k] = Fraction(v) if "/" in v else float(v)
    return out
