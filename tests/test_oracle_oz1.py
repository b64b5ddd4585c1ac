"""Pins for the Scheme I oracle (-m "not gpu").  Each test ties oracle/ to something other
than itself: Python big-int / Fraction arithmetic, numpy's textbook integer matmul, closed
forms and special cases, and the __float128 brute force within the closed-form error bound
(SURVEY 8(c) "What pins each part")."""
import os
from fractions import Fraction

import numpy as np
import pytest

import emugemm_inputs as G
from oracle import oracle as O
from exact_helpers import BETA, max_exp, trunc_scaled, read_golden

GOLD = read_golden(os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt"))


@pytest.fixture(autouse=True, params=["twos", "signmag"])
def digit_form(request):
    """Every pin below runs in both 7-bit digit forms: the default two's-complement digits (R24) and the
    sign-magnitude digits (R1).  Both spell the same integer X = trunc(x 2^(7p)), so the invariants are shared; the two
    pins that describe the digits themselves branch on the form."""
    O.set_slice_bits(7 if request.param == "twos" else O.DIGITS_SIGNMAG)
    yield request.param
    O.set_slice_bits(7)


def test_paper_constants():
    # PAPER.md:88 p(p+1)/2 products; PAPER.md:76 signed slices => beta <= 7
    assert int(GOLD["oz1_product_count_p6"][0]) == 6 * 7 // 2
    assert int(GOLD["oz1_product_count_p8"][0]) == 8 * 9 // 2
    assert O.BETA == int(GOLD["oz1_max_beta_signed"][0]) == BETA


def test_exponents_match_frexp_definition():
    A, B = G.real_pair(9, 7, 33, 2.0, 11)
    A[3, :] = 0.0           # all-zero row -> exponent 0 (R2)
    A[4, 5] = 5e-324        # subnormal handled exactly
    B[:, 2] = 0.0
    eA, eB = O.row_exponents(A), O.col_exponents(B)
    assert [max_exp(A[i]) for i in range(9)] == list(eA)
    assert [max_exp(B[:, j]) for j in range(7)] == list(eB)
    assert eA[3] == 0 and eB[2] == 0


@pytest.mark.parametrize("p", [1, 2, 3, 6, 8])
def test_slices_resum_to_truncated_input(p, digit_form):
    """Invariant: sum_t A'_t 2^(beta(p-1-t)) == sign * trunc(|x| 2^(beta p)), x = a 2^-eA (exact ints)."""
    A, B = G.real_pair(6, 5, 40, 2.0, 5)
    A[0, 0] = 0.0
    A[1, 1] = -A[1].max() * 3  # the row maximum itself, negative
    eA, eB = O.row_exponents(A), O.col_exponents(B)
    SA, SB = O.oz1_slices_rows(A, eA, p), O.oz1_slices_cols(B, eB, p)
    if digit_form == "signmag":
        assert SA.min() >= -127 and SA.max() <= 127 and SB.min() >= -127 and SB.max() <= 127
    else:   # signed leading slice, non-negative remaining slices
        assert SA[0].min() >= -128 and SA[0].max() <= 127 and SB[0].min() >= -128 and SB[0].max() <= 127
        assert p == 1 or (SA[1:].min() >= 0 and SA[1:].max() <= 127 and SB[1:].min() >= 0 and SB[1:].max() <= 127)
    for i in range(A.shape[0]):
        for h in range(A.shape[1]):
            want = trunc_scaled(A[i, h], BETA * p - int(eA[i]))
            got = sum(int(SA[t, i, h]) << (BETA * (p - 1 - t)) for t in range(p))
            assert got == want
            assert abs(want) < (1 << (BETA * p))
    for j in range(B.shape[1]):
        for h in range(B.shape[0]):
            want = trunc_scaled(B[h, j], BETA * p - int(eB[j]))
            got = sum(int(SB[t, j, h]) << (BETA * (p - 1 - t)) for t in range(p))
            assert got == want


def test_slices_match_fp64_digit_recurrence(digit_form):
    """Second derivation: d = trunc(r 2^beta); r = r 2^beta - d in FP64 (exact: power-of-two scalings and subtraction of
    the integer part only) gives the 7-bit fields of |X|: the sign-magnitude digits are sign * field; the two's-complement
    digits are the fields of X = sign * |X| -- for a negative element the fields of 2^(7p + 1) - |X| (borrow propagation from
    the lowest non-zero field), the leading one read as a signed byte."""
    p = 7
    A, _ = G.real_pair(16, 4, 64, 1.0, 9)
    A[2, 3] = -A[2, 3] if A[2, 3] > 0 else A[2, 3]
    eA = O.row_exponents(A)
    SA = O.oz1_slices_rows(A, eA, p)
    r = np.abs(A) * np.exp2(-eA.astype(np.float64))[:, None]
    sgn = np.where(A < 0, -1, 1)
    fields = []
    for t in range(p):
        r = r * 2.0 ** BETA
        d = np.floor(r)
        r = r - d
        fields.append(d.astype(np.int64))
    if digit_form == "signmag":
        for t in range(p):
            assert np.array_equal((sgn * fields[t]).astype(np.int8), SA[t])
        return
    # negate field-wise with borrow, from the least significant field up: -|X| = sum_t d_t 128^(p-1-t), d_t in [0, 127] (t > 0)
    want = [f.copy() for f in fields]
    neg = A < 0
    borrow = np.zeros_like(fields[0])
    for t in range(p - 1, -1, -1):
        v = -fields[t] - borrow                      # in [-128, 0]
        if t > 0:
            borrow = (v < 0).astype(np.int64)
            v = v + 128 * borrow                     # in [0, 127]
        want[t] = np.where(neg, v, fields[t])
    for t in range(p):
        assert np.array_equal(want[t].astype(np.int8), SA[t]), t


def test_row_scaling_changes_only_exponent():
    A, _ = G.real_pair(5, 3, 50, 1.0, 2)
    A2 = A.copy()
    A2[2] *= 2.0 ** 13
    e1, e2 = O.row_exponents(A), O.row_exponents(A2)
    assert e2[2] == e1[2] + 13 and np.array_equal(np.delete(e1, 2), np.delete(e2, 2))
    assert np.array_equal(O.oz1_slices_rows(A, e1, 6), O.oz1_slices_rows(A2, e2, 6))


def test_accumulators_are_textbook_integer_matmul():
    p = 5
    A, B = G.real_pair(17, 13, 70, 0.5, 3)
    eA, eB = O.row_exponents(A), O.col_exponents(B)
    SA, SB = O.oz1_slices_rows(A, eA, p), O.oz1_slices_cols(B, eB, p)
    CS = O.oz1_accumulators(SA, SB)
    for s in range(p):
        ref = sum(SA[t].astype(np.int64) @ SB[s - t].astype(np.int64).T for t in range(s + 1))
        assert np.array_equal(CS[s], ref)
        assert np.abs(CS[s]).max() <= (s + 1) * A.shape[1] * 128 * 128   # |digit| <= 127 (sign-magnitude) / 128 (leading two's-complement digit)


def test_shift_reduce_closed_form_fractions(digit_form):
    """C == product of the truncated operands minus the dropped pairs (t+u >= p), exactly, then
    one rounding; checked with Fractions on a tiny input, with alpha and beta."""
    p = 4
    A, B, Cin = G.real_pair(4, 3, 9, 2.0, 21, with_c=True)
    alpha, beta = 1.75, -0.5
    eA, eB = O.row_exponents(A), O.col_exponents(B)
    got = O.dgemm_oz1(A, B, p, alpha=alpha, beta=beta, Cin=Cin)
    for i in range(4):
        for j in range(3):
            tot = Fraction(0)
            for h in range(9):
                XA = trunc_scaled(A[i, h], BETA * p - int(eA[i]))
                XB = trunc_scaled(B[h, j], BETA * p - int(eB[j]))
                if digit_form == "signmag":   # digits = sign * 7-bit fields of |X|
                    da = [(abs(XA) >> (BETA * (p - 1 - t))) & 127 for t in range(p)]
                    db = [(abs(XB) >> (BETA * (p - 1 - t))) & 127 for t in range(p)]
                    sg = (-1 if XA < 0 else 1) * (-1 if XB < 0 else 1)
                else:                         # two's-complement fields of X itself (Python's >> floors): signed leading digit
                    da = [(XA >> (BETA * (p - 1 - t))) & 127 if t else XA >> (BETA * (p - 1)) for t in range(p)]
                    db = [(XB >> (BETA * (p - 1 - t))) & 127 if t else XB >> (BETA * (p - 1)) for t in range(p)]
                    sg = 1
                for t in range(p):
                    for u in range(p):
                        if t + u < p:  # kept pairs only (Eq. 2)
                            tot += sg * da[t] * db[u] * Fraction(2) ** (-BETA * (t + 1) - BETA * (u + 1))
            val = Fraction(alpha) * tot * Fraction(2) ** (int(eA[i]) + int(eB[j])) + Fraction(beta) * Fraction(float(Cin[i, j]))
            # one correct rounding: float(Fraction) rounds to nearest even
            assert got[i, j] == float(val)


def test_identity_gives_truncated_A():
    """B = I: C = A truncated to beta*p bits below the row exponent, exactly (eB = 1, B'_0 = 64)."""
    p = 6
    A, _ = G.real_pair(12, 12, 12, 1.0, 4)
    C = O.dgemm_oz1(A, np.eye(12), p)
    eA = O.row_exponents(A)
    # identity column: b = 1 = 0.5 * 2^1 -> X_B = 2^(beta p - 1): exact single digit 64 in slice 0,
    # pairs (t, 0) kept for all t < p, so C = trunc(A) exactly.
    for i in range(12):
        for j in range(12):
            want = Fraction(trunc_scaled(A[i, j], BETA * p - int(eA[i]))) * Fraction(2) ** (int(eA[i]) - BETA * p)
            assert C[i, j] == float(want)


def test_small_integers_exact():
    rng = np.random.default_rng(7)
    A = rng.integers(-63, 64, size=(20, 30)).astype(np.float64)
    B = rng.integers(-63, 64, size=(30, 10)).astype(np.float64)
    for p in (2, 3, 8):
        assert np.array_equal(O.dgemm_oz1(A, B, p), A @ B)
    assert np.array_equal(O.sgemm_oz1(A, B, 2).astype(np.float64), A @ B)


def oz1_error_bound(A, B, p):
    """|C - AB|_ij < 2^(eA_i+eB_j-beta p) (sum_h(|x_ih|+|y_hj|) + k(p-1)/(1-2^-beta)) + 1/2 ulp
    (x, y the operands scaled into (-1,1)); SURVEY 8(c)."""
    eA, eB = O.row_exponents(A), O.col_exponents(B)
    x = np.abs(A) * np.exp2(-eA.astype(float))[:, None]
    y = np.abs(B) * np.exp2(-eB.astype(float))[None, :]
    k = A.shape[1]
    term = x.sum(1)[:, None] + y.sum(0)[None, :] + k * (p - 1) / (1 - 2.0 ** -BETA)
    return np.exp2(eA[:, None].astype(float) + eB[None, :] - BETA * p) * term


def test_config0_vs_float128_bruteforce_within_bound():
    """BASELINE config 1 (index 0): 256^3, phi 0.5, seed 0, p = 6, checked against the __float128
    product of the ORIGINAL operands with the closed-form truncation bound."""
    cfg = G.CONFIGS[0]
    (m, n, k), = cfg["shapes"]
    A, B = G.real_pair(m, n, k, cfg["phi"][0], cfg["seed"])
    C = O.dgemm_oz1(A, B, 6)
    exact, absAB = O.bf128_dgemm(A, B)
    err = np.abs(C - exact)
    bound = oz1_error_bound(A, B, 6) + 0.5 * np.spacing(np.abs(exact))
    assert (err < bound).all()
    # the bound is not vacuous: the observed error is a few % of it and a 5-slice run violates nothing
    # but is > 2^5 times worse; a dropped leading pair would exceed the bound by orders of magnitude.
    assert err.max() > 1e-3 * bound.max()
    err5 = np.abs(O.dgemm_oz1(A, B, 5) - exact)
    assert np.median(err5) > 30 * np.median(err)


def test_p8_narrow_range_close_to_correctly_rounded():
    rng = np.random.default_rng(3)
    A = 1.0 + rng.random((24, 40))
    B = 1.0 + rng.random((40, 16))
    C = O.dgemm_oz1(A, B, 8)
    exact, _ = O.bf128_dgemm(A, B)
    assert (np.abs(C - exact) <= 4 * np.spacing(exact)).all()


def test_sgemm_matches_definition_on_float_inputs():
    """FP32 entry: inputs are float32 widened exactly.  Narrow-range rows (all entries within 2x of
    the row max): p = 4 keeps 28 >= 24+1 bits, so with B = I the result is A exactly.  Wide range:
    C = trunc(A) to 28 bits below the row exponent, rounded once to float.  General case: within
    the closed-form bound + 1/2 ulp_f32 of the __float128 product."""
    rng = np.random.default_rng(8)
    An = (1.0 + rng.random((10, 10))).astype(np.float32)
    assert np.array_equal(O.sgemm_oz1(An, np.eye(10, dtype=np.float32), 4), An)
    A, B = G.real_pair(10, 10, 10, 1.0, 8, dtype=np.float32)
    Ct = O.sgemm_oz1(A, np.eye(10, dtype=np.float32), 4)
    eA = O.row_exponents(A.astype(np.float64))
    for i in range(10):
        for j in range(10):
            want = Fraction(trunc_scaled(float(A[i, j]), BETA * 4 - int(eA[i]))) * Fraction(2) ** (int(eA[i]) - BETA * 4)
            assert Ct[i, j] == np.float32(float(want))
    C = O.sgemm_oz1(A, B, 4).astype(np.float64)
    exact, _ = O.bf128_dgemm(A.astype(np.float64), B.astype(np.float64))
    bound = oz1_error_bound(A.astype(np.float64), B.astype(np.float64), 4) + 0.5 * np.spacing(np.abs(exact).astype(np.float32)).astype(np.float64)
    assert (np.abs(C - exact) <= bound).all()


def test_sampled_equals_full():
    A, B = G.real_pair(40, 36, 64, 2.0, 12)
    rows, cols = np.array([0, 7, 39]), np.array([1, 35])
    full = O.dgemm_oz1(A, B, 7)
    assert np.array_equal(O.oz1_sampled(A, B, 7, rows, cols), full[np.ix_(rows, cols)])


def test_k_zero_and_empty():
    A = np.zeros((3, 0)); B = np.zeros((0, 2)); Cin = np.ones((3, 2))
    assert np.array_equal(O.dgemm_oz1(A, B, 4, alpha=1.0, beta=2.0, Cin=Cin), 2 * Cin)
