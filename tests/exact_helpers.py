"""Independent exact arithmetic for pinning the oracle: Python ints / Fractions only.
Nothing here calls oracle/ or the CUDA path."""
import math
from fractions import Fraction

BETA = 7


def frexp_exp(a):
    """e with |a| in [2^(e-1), 2^e); None for 0."""
    if a == 0:
        return None
    return math.frexp(a)[1]


def max_exp(values):
    es = [frexp_exp(float(v)) for v in values if v != 0]
    return max(es) if es else 0


def trunc_scaled(a, shift):
    """trunc(a * 2^shift) toward zero as a Python int, exactly."""
    f = Fraction(float(a)) * (Fraction(2) ** shift)
    q = abs(f.numerator) // f.denominator
    return q if f >= 0 else -q


def sym(x, m):
    r = x % m  # Python: floored, in [0, m)
    if r >= (m + 1) // 2:
        r -= m
    return r


def greedy_moduli(n):
    out = []
    c = 256
    while len(out) < n:
        if all(math.gcd(c, q) == 1 for q in out):
            out.append(c)
        c -= 1
    return out


def read_golden(path):
    vals = {}
    for line in open(path):
        line = line.split("#")[0].strip()
        if "=" in line:
            k, v = line.split("=")
            vals[k.strip()] = v.split()
    return vals
