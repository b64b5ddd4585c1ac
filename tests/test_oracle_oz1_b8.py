"""Pins for the 8-bit slice mode of the Scheme I oracle (-m "not gpu"): balanced signed base-256 digits
(R23; "slices of beta <= 8 bits").  Same structure as
test_oracle_oz1.py: exact Python integers / Fractions, numpy integer matmul, special cases, __float128
brute force inside a bound written out here."""
from fractions import Fraction

import numpy as np
import pytest

import emugemm_inputs as G
from oracle import oracle as O
from exact_helpers import trunc_scaled


@pytest.fixture(autouse=True)
def balanced_mode():
    O.set_slice_bits(8)
    yield
    O.set_slice_bits(7)


@pytest.mark.parametrize("p", [1, 2, 3, 7, 8])
def test_digits_resum_to_truncated_input(p):
    """sum_t d_t 256^(p-1-t) == trunc(a 2^(8p - e - 2)) exactly, d_t in [-128, 127], |X| < 2^(8p-2)."""
    A, B = G.real_pair(6, 5, 40, 2.0, 5)
    A[0, 0] = 0.0
    A[1, 1] = -np.abs(A[1]).max() * 3   # the row maximum itself, negative
    A[2, 2] = np.abs(A[2]).max() * 1.999  # and one just below the next power of two, positive
    eA, eB = O.row_exponents(A), O.col_exponents(B)
    SA, SB = O.oz1_slices_rows(A, eA, p), O.oz1_slices_cols(B, eB, p)
    assert SA.min() >= -128 and SA.max() <= 127
    for i in range(A.shape[0]):
        for h in range(A.shape[1]):
            want = trunc_scaled(A[i, h], 8 * p - int(eA[i]) - 2)
            got = sum(int(SA[t, i, h]) * 256 ** (p - 1 - t) for t in range(p))
            assert got == want and abs(want) < (1 << (8 * p - 2))
    for j in range(B.shape[1]):
        for h in range(B.shape[0]):
            want = trunc_scaled(B[h, j], 8 * p - int(eB[j]) - 2)
            assert sum(int(SB[t, j, h]) * 256 ** (p - 1 - t) for t in range(p)) == want


def test_digits_are_the_unique_balanced_expansion():
    """Second derivation in Python integers: repeatedly take the residue in [-128, 127] from the low end."""
    p = 7
    A, _ = G.real_pair(8, 4, 32, 1.0, 9)
    eA = O.row_exponents(A)
    SA = O.oz1_slices_rows(A, eA, p)
    for i in range(8):
        for h in range(32):
            X = trunc_scaled(A[i, h], 8 * p - int(eA[i]) - 2)
            for t in reversed(range(p)):
                d = ((X + 128) % 256) - 128
                assert int(SA[t, i, h]) == d
                X = (X - d) // 256
            assert X == 0


def test_closed_form_with_fractions():
    """C == sum over the KEPT digit pairs (t + u < p) of the exact digit products, one rounding; alpha, beta."""
    p = 3
    A, B, Cin = G.real_pair(4, 3, 9, 2.0, 21, with_c=True)
    alpha, beta = 1.75, -0.5
    eA, eB = O.row_exponents(A), O.col_exponents(B)
    SA, SB = O.oz1_slices_rows(A, eA, p), O.oz1_slices_cols(B, eB, p)
    got = O.dgemm_oz1(A, B, p, alpha=alpha, beta=beta, Cin=Cin)
    for i in range(4):
        for j in range(3):
            tot = Fraction(0)
            for h in range(9):
                for t in range(p):
                    for u in range(p - t):
                        tot += int(SA[t, i, h]) * int(SB[u, j, h]) * Fraction(256) ** (-(t + 1) - (u + 1))
            val = Fraction(alpha) * tot * Fraction(2) ** (int(eA[i]) + 2 + int(eB[j]) + 2) + Fraction(beta) * Fraction(float(Cin[i, j]))
            assert got[i, j] == float(val)


def test_accumulators_are_textbook_integer_matmul_and_bounded():
    p = 5
    A, B = G.real_pair(17, 13, 70, 0.5, 3)
    eA, eB = O.row_exponents(A), O.col_exponents(B)
    SA, SB = O.oz1_slices_rows(A, eA, p), O.oz1_slices_cols(B, eB, p)
    CS = O.oz1_accumulators(SA, SB)
    for s in range(p):
        ref = sum(SA[t].astype(np.int64) @ SB[s - t].astype(np.int64).T for t in range(s + 1))
        assert np.array_equal(CS[s], ref)
        assert np.abs(CS[s]).max() <= (s + 1) * A.shape[1] * 128 * 128


def test_small_integers_exact_and_identity():
    rng = np.random.default_rng(7)
    A = rng.integers(-31, 32, size=(20, 30)).astype(np.float64)
    B = rng.integers(-31, 32, size=(30, 10)).astype(np.float64)
    for p in (2, 3, 7):
        assert np.array_equal(O.dgemm_oz1(A, B, p), A @ B)
    # B = I: C = A truncated to 8p - 2 bits below the row exponent (the single digit of 1 is 32 in slice 0)
    p = 6
    A, _ = G.real_pair(12, 12, 12, 1.0, 4)
    C = O.dgemm_oz1(A, np.eye(12), p)
    eA = O.row_exponents(A)
    for i in range(12):
        for j in range(12):
            want = Fraction(trunc_scaled(A[i, j], 8 * p - int(eA[i]) - 2)) * Fraction(2) ** (int(eA[i]) + 2 - 8 * p)
            assert C[i, j] == float(want)


def b8_error_bound(A, B, p):
    """With x = a 2^-(eA+2), y = b 2^-(eB+2) in (-1/4, 1/4): truncation |x - x_p| < 256^-p, and the dropped digit
    pairs (t + u >= p) are bounded by sum_{s >= p} min(s + 1, p) 128^2 256^-(s+2) < p 128^2 256^-(p+2) / (1 - 1/256):
    |C - AB|_ij < 2^(eA+eB+4) [ 256^-p sum_h(|x| + |y|) + k p 2^14 256^-(p+2) (256/255) ] + 1/2 ulp."""
    eA, eB = O.row_exponents(A), O.col_exponents(B)
    x = np.abs(A) * np.exp2(-(eA + 2).astype(float))[:, None]
    y = np.abs(B) * np.exp2(-(eB + 2).astype(float))[None, :]
    k = A.shape[1]
    term = 256.0 ** -p * (x.sum(1)[:, None] + y.sum(0)[None, :]) + k * p * 2.0 ** 14 * 256.0 ** -(p + 2) * 256 / 255
    return np.exp2(eA[:, None].astype(float) + eB[None, :] + 4) * term


@pytest.mark.parametrize("p", [3, 5, 7])
def test_vs_float128_bruteforce_within_bound(p):
    A, B = G.real_pair(96, 80, 128, 0.5, 0)
    C = O.dgemm_oz1(A, B, p)
    exact, _ = O.bf128_dgemm(A, B)
    err = np.abs(C - exact)
    bound = b8_error_bound(A, B, p) + 0.5 * np.spacing(np.abs(exact))
    assert (err < bound).all()
    assert err.max() > 1e-4 * bound.max()  # not vacuous


def test_seven_balanced_slices_match_eight_signmagnitude_slices_in_accuracy():
    """8 bits x 7 slices (28 products) reaches the accuracy of 7 bits x 8 slices (36 products): the point of f1."""
    A, B = G.real_pair(64, 64, 256, 0.5, 1)
    exact, absAB = O.bf128_dgemm(A, B)
    e8 = np.abs(O.dgemm_oz1(A, B, 7) - exact) / absAB
    O.set_slice_bits(7)
    e7 = np.abs(O.dgemm_oz1(A, B, 8) - exact) / absAB
    assert e8.max() < 4 * e7.max() and e8.max() < 2.0 ** -44


def test_sampled_equals_full():
    A, B = G.real_pair(40, 30, 64, 1.0, 8)
    full = O.dgemm_oz1(A, B, 7)
    rows, cols = np.array([0, 5, 39]), np.array([1, 29])
    assert np.array_equal(O.oz1_sampled(A, B, 7, rows, cols), full[np.ix_(rows, cols)])
