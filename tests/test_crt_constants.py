"""not-gpu: the host-side constants of the exact FP64 CRT kernel (csrc/crt.cu, R17) against Python big
integers and the oracle's CRT (Eq. 8).

The kernel's arithmetic is re-stated here over Python integers, step for step (pair combination of the biased
bytes, balanced-digit accumulators, quotient, carry normalisation), with the library's own constants: the result
must equal the oracle's big-integer CRT for every residue vector, and every intermediate must stay inside the
53-bit window that makes the device FMAs exact."""
import numpy as np
import pytest

import paper_2606_25453_b200 as E
from paper_2606_25453_b200 import binding as Bn
from oracle import oracle as O


def _val(digits, g):
    return sum(d << (j * g) if d >= 0 else -((-d) << (j * g)) for j, d in enumerate(digits))


@pytest.mark.parametrize("N", list(range(2, 21)))
def test_constants_are_the_crt_weights(N):
    c = Bn.crt_constants(N)
    mods = [int(x) for x in O.oz2_moduli(N)]
    P = O.oz2_P(N)
    g, J, NP = c["digit_bits"], c["n_digits"], c["n_pairs"]
    assert NP == (N + 1) // 2
    assert J * g >= P.bit_length() + 1
    assert _val(c["P"], g) == P
    xsum = 0
    for q in range(NP):
        m1 = mods[2 * q]
        m2 = mods[2 * q + 1] if 2 * q + 1 < N else 1
        M, K1, K2, C0, magic = c["pair"][q]
        assert M == m1 * m2 and K1 < 1 << 16 and K2 < 1 << 16
        assert K1 % m1 == 1 % m1 and K1 % m2 == 0 and (m2 == 1 or (K2 % m2 == 1 and K2 % m1 == 0))
        assert C0 % M == 0 and (1 << 24) <= C0 < (1 << 24) + M and magic == (1 << 32) // M
        W = _val(c["W"][q], g)
        assert 0 < W < P and W % M == 1 and W % (P // M) == 0   # the CRT weight of the pair modulus
        xsum += M - 1
        for d in c["W"][q]:
            assert abs(d) <= 1 << (g - 1)
    for d in c["P"]:
        assert abs(d) <= 1 << (g - 1)
    assert ((xsum + 2) << g) <= 1 << 52   # every accumulator, Q P_j and T_j stay exact in FP64


def _device_algorithm(c, mods, res):
    """The kernel's steps over Python integers; returns (C', max |intermediate|)."""
    g, J, NP = c["digit_bits"], c["n_digits"], c["n_pairs"]
    N = len(mods)
    acc = [0] * J
    big = 0
    for q in range(NP):
        M, K1, K2, C0, magic = c["pair"][q]
        c1 = int(res[2 * q])
        c2 = int(res[2 * q + 1]) if 2 * q + 1 < N else 0
        s = K1 * c1 + K2 * c2 + C0
        assert 0 < s < 1 << 26
        x = s - ((s * magic) >> 32) * M
        assert 0 <= x < 2 * M
        x = min(x, (x - M) % (1 << 32))
        assert x == s % M and x % mods[2 * q] == c1 % mods[2 * q]
        for j in range(J):
            acc[j] += c["W"][q][j] * x
            big = max(big, abs(acc[j]))
    P = _val(c["P"], g)
    # the kernel takes the quotient from the two leading digits only
    top = acc[J - 1] * (1 << ((J - 1) * g)) + (acc[J - 2] * (1 << ((J - 2) * g)) if J > 1 else 0)
    Q = (2 * top + P) // (2 * P)
    S = _val(acc, g)
    assert abs(S - Q * P) <= P // 2 or abs(O.oz2_crt_int(np.array(res, np.int32))) >= P // 4
    T = [acc[j] - Q * c["P"][j] for j in range(J)]
    big = max([big] + [abs(t) for t in T])
    for j in range(J - 1):       # carry normalisation to balanced digits
        carry = (T[j] + (1 << (g - 1))) >> g
        T[j] -= carry << g
        T[j + 1] += carry
        big = max(big, abs(T[j + 1]))
        assert abs(T[j]) <= 1 << (g - 1)
    return _val(T, g), big


@pytest.mark.parametrize("N", [2, 3, 8, 11, 12, 14, 15, 16, 18, 19, 20])
def test_integer_restatement_matches_oracle_crt(N):
    c = Bn.crt_constants(N)
    mods = [int(x) for x in O.oz2_moduli(N)]
    P = O.oz2_P(N)
    rng = np.random.default_rng(N)
    cases = []
    lo = [-(m // 2) if m % 2 == 0 else -((m - 1) // 2) for m in mods]
    hi = [(m // 2) - 1 if m % 2 == 0 else (m - 1) // 2 for m in mods]
    cases.append(lo); cases.append(hi); cases.append([0] * N)
    for X in (1, -1, 127, -128, P // 4 - 1, -(P // 4) + 1, 12345678901234567890 % (P // 4)):
        cases.append([((X % m) + m) % m for m in mods])
    for _ in range(200):
        X = int(rng.integers(-2**62, 2**62)) * int(rng.integers(1, 2**62)) % (P // 2) - P // 4
        cases.append([X % m for m in mods])
    for res in cases:
        sym = [r - m if r >= (m + 1) // 2 else r for r, m in zip(res, mods)]   # symmetric INT8 residues (R11)
        want = O.oz2_crt_int(np.array(sym, np.int32))
        got, big = _device_algorithm(c, mods, sym)
        # lo / hi vectors are arbitrary residues: the true value may lie beyond P/4, then only congruence holds
        if abs(want) < P // 4:
            assert got == want
        else:
            assert (got - want) % P == 0
        assert big < 1 << 52
