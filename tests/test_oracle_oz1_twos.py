"""not-gpu: oracle pins for the DEFAULT digit form of Scheme I, two's-complement 7-bit digits (R24; "a signed leading
slice with unsigned remaining slices", here at beta = 7 so that every slice is an INT8 value).

What is fixed by the mathematics: the digits are the two's-complement fields of the SAME integer X = trunc(x 2^(7p))
that the sign-magnitude digits of R1 spell, so (a) sum_t d_t 2^(7(p-1-t)) == X for both forms, (b) d_0 is the only
digit that can be negative and the others lie in [0, 127], (c) a non-negative element has the same digits in both forms,
(d) whenever the dropped pairs vanish (small integer operands) both forms give the same, exact, product,
(e) the full product stays within the method's error bound of the exact product."""
from fractions import Fraction

import numpy as np
import pytest

import emugemm_inputs as G
from oracle import oracle as O


@pytest.fixture()
def twos():
    O.set_slice_bits(7)      # the default form (R24)
    yield
    O.set_slice_bits(7)


def _X(a, e, p):
    """trunc(a 2^(7p - e)) toward zero, exactly, with Python integers (R1 / R3)."""
    f = Fraction(float(a)) * Fraction(2) ** (7 * p - int(e))
    n = abs(f.numerator) // f.denominator
    return n if f >= 0 else -n


@pytest.mark.parametrize("p", [1, 2, 3, 5, 8])
def test_digits_are_the_twos_complement_fields_of_the_same_integer(twos, p):
    A, _ = G.real_pair(37, 5, 61, 2.0, 11)
    A[0, 0] = 0.0
    A[1, :] = -np.abs(A[1, :])                       # an all-negative row
    A[2, 3] = -np.abs(A[2]).max() * 1.999            # the row maximum is negative and nearly 2^e
    A[3, 1] = np.abs(A[3]).max() * 1.999
    A[4, 7] = -2.0 ** -60 * np.abs(A[4]).max()       # a tiny negative value: X = 0 or -0 -> digits all zero (trunc toward zero)
    eA = O.row_exponents(A)
    S = O.oz1_slices_rows(A, eA, p).astype(np.int64)          # [p][m][k]
    O.set_slice_bits(O.DIGITS_SIGNMAG)
    S1 = O.oz1_slices_rows(A, eA, p).astype(np.int64)
    O.set_slice_bits(7)
    assert S[0].min() >= -128 and S[0].max() <= 127
    if p > 1:
        assert S[1:].min() >= 0 and S[1:].max() <= 127           # every slice but the leading one is sign-free
    w = np.array([1 << (7 * (p - 1 - t)) for t in range(p)], dtype=object)
    for i in range(A.shape[0]):
        for h in range(A.shape[1]):
            X = _X(A[i, h], eA[i], p)
            assert sum(int(S[t, i, h]) * int(w[t]) for t in range(p)) == X      # (a) two's complement
            assert sum(int(S1[t, i, h]) * int(w[t]) for t in range(p)) == X     # (a) sign-magnitude: the same integer
            if A[i, h] >= 0:
                assert all(S[t, i, h] == S1[t, i, h] for t in range(p))         # (c)
    assert (S[:, 4, 7] == 0).all()                                              # trunc toward zero: a tiny negative is 0, not -1


def test_columns_match_rows_of_the_transpose(twos):
    A, B = G.real_pair(9, 13, 40, 1.0, 3)
    eB = O.col_exponents(B)
    SB = O.oz1_slices_cols(B, eB, 6)
    SBt = O.oz1_slices_rows(np.ascontiguousarray(B.T), O.row_exponents(np.ascontiguousarray(B.T)), 6)
    assert np.array_equal(SB, SBt)


def test_small_integer_operands_are_exact_in_both_forms(twos):
    """Integers below 2^7: X = a 2^(7p - e) is a multiple of 2^(7(p-1)), so in BOTH forms only the leading digit is
    non-zero (the two's complement of a multiple of 2^j is a multiple of 2^j), no kept or dropped pair involves a lower
    digit and the product is exact for every p."""
    rng = np.random.default_rng(5)
    A = rng.integers(-127, 128, size=(20, 33)).astype(np.float64)
    B = rng.integers(-127, 128, size=(33, 17)).astype(np.float64)
    want = A @ B
    for p in (1, 2, 4, 8):
        S = O.oz1_slices_rows(A, O.row_exponents(A), p)
        assert (S[1:] == 0).all()
        assert np.array_equal(O.dgemm_oz1(A, B, p), want), p
        O.set_slice_bits(O.DIGITS_SIGNMAG)
        r1 = O.dgemm_oz1(A, B, p)
        O.set_slice_bits(7)
        assert np.array_equal(r1, want)


@pytest.mark.parametrize("p", [3, 6, 8])
def test_error_bound_against_the_exact_product(twos, p):
    """Against the __float128 brute force: the dropped pairs t + u >= p and the truncation of the operands bound the error by
    (k (p + 1) 2^(-7p + 2) + 2^-52) 2^(eA_i + eB_j) -- each dropped pair is below 2^(-7(t+u)) * 128 * 128 / 2^14 per term."""
    A, B = G.real_pair(31, 23, 200, 0.5, 9)
    exact, _ = O.bf128_dgemm(A, B)
    got = O.dgemm_oz1(A, B, p)
    eA, eB = O.row_exponents(A), O.col_exponents(B)
    scale = np.exp2(eA.astype(np.float64))[:, None] * np.exp2(eB.astype(np.float64))[None, :]
    bound = (200 * (p + 1) * 2.0 ** (-7 * p + 2) + 2.0 ** -52) * scale
    assert (np.abs(got - exact) <= bound).all()
    O.set_slice_bits(O.DIGITS_SIGNMAG)
    r1 = O.dgemm_oz1(A, B, p)
    O.set_slice_bits(7)
    assert (np.abs(got - r1) <= 2 * bound).all()     # the two digit forms differ only by their dropped pairs
    if p == 8:
        assert np.abs(got - exact).max() <= 4 * np.abs(exact).max() * 2.0 ** -45
