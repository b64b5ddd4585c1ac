"""Pins for the Scheme II oracle (-m "not gpu"): Python big integers are the independent
reference (SURVEY 8(c) "What pins each part")."""
import math
import os

import numpy as np
import pytest

import emugemm_inputs as G
from oracle import oracle as O
from exact_helpers import greedy_moduli, max_exp, read_golden, sym, trunc_scaled

GOLD = read_golden(os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt"))


def test_moduli_paper_and_coprime():
    mod = [int(x) for x in O.oz2_moduli(24)]
    assert mod[:3] == [int(x) for x in GOLD["moduli_first_three"]]
    assert mod == greedy_moduli(24)
    assert all(m <= 256 for m in mod) and mod == sorted(mod, reverse=True)
    for i in range(24):
        for j in range(i):
            assert math.gcd(mod[i], mod[j]) == 1
    for N in (2, 12, 20, 24):
        assert O.oz2_P(N) == math.prod(mod[:N])


@pytest.mark.parametrize("N", [2, 8, 12, 16, 20, 24])
def test_crt_weights(N):
    mod = greedy_moduli(N)
    P = math.prod(mod)
    w = O.oz2_weights(N)
    for l, m in enumerate(mod):
        assert w[l] == (P // m) * pow(P // m, -1, m)  # Eq. 8: (P/m_l) q_l
        assert w[l] % m == 1
        for j, mj in enumerate(mod):
            if j != l:
                assert w[l] % mj == 0


@pytest.mark.parametrize("N", [2, 12, 14, 18, 20, 24])
def test_crt_round_trip(N):
    mod = greedy_moduli(N)
    P = math.prod(mod)
    rng = np.random.default_rng(N)
    xs = [0, 1, -1, P // 2, -(P // 2) + (1 - P % 2), (P - 1) // 2, -((P - 1) // 2)]
    xs += [int.from_bytes(rng.bytes(24), "little") % P - P // 2 for _ in range(200)]
    for x in xs:
        if not (-P / 2 < x <= P / 2):
            continue
        c = [sym(x, m) for m in mod]
        assert O.oz2_crt_int(c) == x
        # any representative of the residue class gives the same X
        assert O.oz2_crt_int([ci + m for ci, m in zip(c, mod)]) == x


def test_budget_rule():
    """T = max{T: k 2^(T+2) <= P} (3M: T+3); values listed in SURVEY 8(c) step 2."""
    want = {12: (40, 39), 14: (48, 47), 16: (55, 55), 18: (63, 62), 20: (70, 70)}
    for N, (a, b) in want.items():
        T, tA, tB = O.oz2_budget(N, 8192)
        P = math.prod(greedy_moduli(N))
        assert 8192 * 2 ** (T + 2) <= P < 8192 * 2 ** (T + 3)
        assert (tA, tB) == (a, b) and tA + tB == T
    assert O.oz2_budget(14, 8192, True)[1:] == (47, 47)
    assert O.oz2_budget(18, 8192, True)[1:] == (62, 62)
    assert O.oz2_budget(14, 4096, True)[1:] == (48, 47)
    assert O.oz2_budget(18, 4096, True)[1:] == (63, 62)
    for N, k in ((12, 1), (20, 100000), (16, 777)):
        T, _, _ = O.oz2_budget(N, k, True)
        P = math.prod(greedy_moduli(N))
        assert k * 2 ** (T + 3) <= P < k * 2 ** (T + 4)
    # soft pin: SGEMM runs at 8-11 moduli, DGEMM at 12-15: operand bits at the range
    # starts reach FP32 / approach FP64 significands at k = 8192
    lo_s = int(GOLD["oz2_sgemm_moduli_range"][0]); hi_d = int(GOLD["oz2_dgemm_moduli_range"][1])
    assert O.oz2_budget(lo_s, 8192)[2] >= 24 and O.oz2_budget(hi_d, 8192)[2] >= 51


def test_residues_vs_python_bigint():
    N = 20
    A, B = G.real_pair(5, 4, 30, 1.0, 2)
    A[0, 0] = 0.0
    _, tA, tB = O.oz2_budget(N, 30)
    assert tA > 62  # exercises > 64-bit integers
    eA, eB = O.row_exponents(A), O.col_exponents(B)
    RA, RB = O.oz2_residues_rows(A, eA, tA, N), O.oz2_residues_cols(B, eB, tB, N)
    mod = greedy_moduli(N)
    for l, m in enumerate(mod):
        for i in range(5):
            for h in range(30):
                ai = trunc_scaled(A[i, h], tA - int(eA[i]))
                assert abs(ai) < 2 ** tA
                assert RA[l, i, h] == sym(ai, m)
        for j in range(4):
            for h in range(30):
                assert RB[l, j, h] == sym(trunc_scaled(B[h, j], tB - int(eB[j])), m)
    assert RA[0].min() >= -128 and RA[0].max() <= 127  # m = 256 range (R11)
    for l, m in enumerate(mod[1:], 1):
        assert RA[l].min() >= -(m - 1) // 2 and RA[l].max() <= (m - 1) // 2


def test_modprod_is_integer_matmul_then_sym():
    N = 6
    rng = np.random.default_rng(0)
    RA = rng.integers(-128, 128, size=(N, 9, 50)).astype(np.int8)
    RB = rng.integers(-128, 128, size=(N, 7, 50)).astype(np.int8)
    CR, mx, ACC = O.oz2_modprod(RA, RB, want_acc=True)
    mod = greedy_moduli(N)
    for l, m in enumerate(mod):
        ref = RA[l].astype(np.int64) @ RB[l].astype(np.int64).T
        assert np.array_equal(ACC[l], ref)
        assert np.array_equal(CR[l], np.vectorize(lambda x: sym(int(x), m))(ref).astype(np.int8))
    assert mx == np.abs(ACC).max() < 2 ** 31


@pytest.mark.parametrize("N", [8, 12, 16, 20])
def test_crt_recovers_exact_integer_product(N):
    """X == sum_h a' b' exactly, and the exactness condition 4 sum |a'||b'| < P holds (R12)."""
    m, n, k = 6, 5, 40
    A, B = G.real_pair(m, n, k, 1.0, N)
    _, tA, tB = O.oz2_budget(N, k)
    eA, eB = O.row_exponents(A), O.col_exponents(B)
    RA, RB = O.oz2_residues_rows(A, eA, tA, N), O.oz2_residues_cols(B, eB, tB, N)
    CR, _, _ = O.oz2_modprod(RA, RB)
    P = math.prod(greedy_moduli(N))
    for i in range(m):
        for j in range(n):
            ai = [trunc_scaled(A[i, h], tA - int(eA[i])) for h in range(k)]
            bi = [trunc_scaled(B[h, j], tB - int(eB[j])) for h in range(k)]
            assert 4 * sum(abs(x) * abs(y) for x, y in zip(ai, bi)) < P
            assert O.oz2_crt_int(CR[:, i, j]) == sum(x * y for x, y in zip(ai, bi))


def oz2_error_bound(A, B, tA, tB):
    """|C - AB|_ij <= k 2^(eA_i+eB_j) (2^-tA + 2^-tB + 2^(-tA-tB)) (+ 1/2 ulp), SURVEY 8(c)."""
    eA, eB = O.row_exponents(A), O.col_exponents(B)
    k = A.shape[1]
    return k * np.exp2(eA[:, None].astype(float) + eB[None, :]) * (2.0 ** -tA + 2.0 ** -tB + 2.0 ** (-tA - tB))


@pytest.mark.parametrize("N", [12, 16, 20])
def test_dgemm_oz2_vs_float128_within_bound(N):
    A, B = G.real_pair(48, 40, 96, 1.0, 2)
    _, tA, tB = O.oz2_budget(N, 96)
    C = O.dgemm_oz2(A, B, N)
    exact, _ = O.bf128_dgemm(A, B)
    assert (np.abs(C - exact) <= oz2_error_bound(A, B, tA, tB) + 0.5 * np.spacing(np.abs(exact))).all()
    if N == 12:  # not vacuous: truncation error is visible at 40 bits
        assert np.abs(C - exact).max() > 1e-4 * oz2_error_bound(A, B, tA, tB).max()


def test_dgemm_oz2_correctly_rounded_when_integers_are_exact():
    """Narrow-range input (entries in [1,2)), tA, tB >= 53: a', b' hold every bit, the integer
    product is exact, so C is the correctly rounded A B (== rounded __float128 product)."""
    rng = np.random.default_rng(1)
    A = 1.0 + rng.random((12, 20)); B = 1.0 + rng.random((20, 9))
    _, tA, tB = O.oz2_budget(18, 20)
    assert tA >= 54 and tB >= 54
    exact, _ = O.bf128_dgemm(A, B)
    assert np.array_equal(O.dgemm_oz2(A, B, 18), exact)
    al, be = 0.75, 3.0
    Cin = rng.standard_normal((12, 9))
    got = O.dgemm_oz2(A, B, 18, alpha=al, beta=be, Cin=Cin)
    from fractions import Fraction
    for i in range(12):
        for j in range(9):
            ex = sum(Fraction(float(A[i, h])) * Fraction(float(B[h, j])) for h in range(20))
            assert got[i, j] == float(Fraction(al) * ex + Fraction(be) * Fraction(float(Cin[i, j])))


def test_3m_equals_four_product_complex_integer_matmul():
    """X_re == sum(ar br - ai bi), X_im == sum(ar bi + ai br) exactly in integers (Eq. 16 + R15, R16)."""
    N, m, n, k = 14, 4, 5, 24
    A, B = G.complex_pair(m, n, k, 1.0, 3)
    _, tA, tB = O.oz2_budget(N, k, True)
    eA, eB = O.row_exponents_z(A), O.col_exponents_z(B)
    assert [max_exp(list(A[i].real) + list(A[i].imag)) for i in range(m)] == list(eA)
    assert [max_exp(list(B[:, j].real) + list(B[:, j].imag)) for j in range(n)] == list(eB)
    RA3 = O.oz2_residues_z(A, eA, tA, N, by_cols=False)
    RB3 = O.oz2_residues_z(B, eB, tB, N, by_cols=True)
    mod = greedy_moduli(N)
    for l, mm in enumerate(mod):  # Sigma plane = sym(re + im)
        s = RA3[0, l].astype(int) + RA3[1, l].astype(int)
        assert np.array_equal(RA3[2, l], np.vectorize(lambda x: sym(int(x), mm))(s).astype(np.int8))
    CZ = O.oz2_modprod_3m(RA3, RB3)
    P = math.prod(mod)
    for i in range(m):
        for j in range(n):
            ar = [trunc_scaled(A[i, h].real, tA - int(eA[i])) for h in range(k)]
            ai = [trunc_scaled(A[i, h].imag, tA - int(eA[i])) for h in range(k)]
            br = [trunc_scaled(B[h, j].real, tB - int(eB[j])) for h in range(k)]
            bi = [trunc_scaled(B[h, j].imag, tB - int(eB[j])) for h in range(k)]
            xre = sum(a * b - c * d for a, b, c, d in zip(ar, br, ai, bi))
            xim = sum(a * d + c * b for a, b, c, d in zip(ar, br, ai, bi))
            assert 2 * abs(xre) < P and 2 * abs(xim) < P
            assert O.oz2_crt_int(CZ[0, :, i, j]) == xre
            assert O.oz2_crt_int(CZ[1, :, i, j]) == xim


def test_zgemm_3m_vs_float128():
    N = 18
    A, B, Cin = G.complex_pair(16, 12, 64, 1.0, 3, with_c=True)
    _, tA, tB = O.oz2_budget(N, 64, True)
    exact, absZ = O.bf128_zgemm(A, B)
    C = O.zgemm_oz2_3m(A, B, N)
    eA, eB = O.row_exponents_z(A), O.col_exponents_z(B)
    bound = 2 * 64 * np.exp2(eA[:, None].astype(float) + eB[None, :]) * (2.0 ** -tA + 2.0 ** -tB + 2.0 ** (-tA - tB))
    assert (np.abs(C.real - exact.real) <= bound + np.spacing(np.abs(exact.real))).all()
    assert (np.abs(C.imag - exact.imag) <= bound + np.spacing(np.abs(exact.imag))).all()
    # complex alpha / beta
    al, be = 0.5 - 2j, 1.5 + 0.25j
    C2 = O.zgemm_oz2_3m(A, B, N, alpha=al, beta=be, Cin=Cin)
    ref = al * C + be * Cin
    assert np.allclose(C2, ref, rtol=1e-13, atol=1e-13 * absZ.max())


def test_sampled_equals_full_oz2():
    A, B = G.real_pair(20, 18, 50, 1.0, 5)
    rows, cols = np.array([0, 19]), np.array([3, 17])
    assert np.array_equal(O.oz2_sampled(A, B, 14, rows, cols), O.dgemm_oz2(A, B, 14)[np.ix_(rows, cols)])
    Az, Bz = G.complex_pair(8, 9, 30, 1.0, 6)
    assert np.array_equal(O.oz2_sampled(Az, Bz, 14, rows[:1], cols[:1], is3m=True), O.zgemm_oz2_3m(Az, Bz, 14)[np.ix_(rows[:1], cols[:1])])


# ---- Scheme II on FP32 inputs ("EmuGEMM-II SGEMM (p8-p11)") ----
def test_sgemm_oz2_is_correctly_rounded_when_the_budget_covers_the_inputs():
    """k = 64, N = 10: tA = tB >= 24 + the spread of a narrow-range row, so the integer product is the exact
    product of the float inputs and the result is the correctly rounded float of A.B (float64 matmul of
    24-bit inputs with k = 64 is exact enough to round to the same float except at ties: compare via
    __float128 brute force)."""
    rng = np.random.default_rng(5)
    A = (1.0 + rng.random((24, 64))).astype(np.float32)
    B = (1.0 + rng.random((64, 16))).astype(np.float32)
    T, tA, tB = O.oz2_budget(10, 64)
    assert tA >= 25 and tB >= 25
    C = O.sgemm_oz2(A, B, 10)
    exact, _ = O.bf128_dgemm(A.astype(np.float64), B.astype(np.float64))
    assert np.array_equal(C, exact.astype(np.float32))


def test_sgemm_oz2_small_integers_and_alpha_beta():
    rng = np.random.default_rng(7)
    A = rng.integers(-63, 64, size=(20, 30)).astype(np.float32)
    B = rng.integers(-63, 64, size=(30, 10)).astype(np.float32)
    Cin = rng.integers(-5, 6, size=(20, 10)).astype(np.float32)
    want = 2.0 * (A.astype(np.float64) @ B.astype(np.float64)) - 3.0 * Cin
    assert np.array_equal(O.sgemm_oz2(A, B, 8, alpha=2.0, beta=-3.0, Cin=Cin), want.astype(np.float32))


def test_sgemm_oz2_matches_dgemm_oz2_rounded_once():
    """Same integers as the FP64 entry point on the widened inputs: the float result is within one float ulp of the
    rounded double result (double rounding) and inside the method's bound against the exact product."""
    A, B = G.real_pair(40, 30, 200, 1.0, 3, dtype=np.float32)
    C32 = O.sgemm_oz2(A, B, 9)
    C64 = O.dgemm_oz2(A.astype(np.float64), B.astype(np.float64), 9)
    assert (np.abs(C32.astype(np.float64) - C64) <= np.spacing(np.abs(C64).astype(np.float32)).astype(np.float64)).all()


def test_crt_X_hook_is_exact_beyond_128_bits():
    """The test hook that returns the reconstructed integer must not truncate: |X| up to P/4 ~ 2^154 at N = 20."""
    N = 20
    mods = [int(x) for x in O.oz2_moduli(N)]
    P = O.oz2_P(N)
    Xs = [P // 4 - 1, -(P // 4) + 3, 12345, -1, 0, 2 ** 140 + 7]
    CR = np.empty((N, 2, 3), np.int8)
    for l, m in enumerate(mods):
        r = np.array([x % m for x in Xs])
        CR[l] = np.where(r >= (m + 1) // 2, r - m, r).reshape(2, 3)
    out, Xi = O.oz2_crt(CR, np.zeros(2, np.int32), np.zeros(3, np.int32), 0, 0, want_X=True)
    assert sum(Xi, []) == Xs
    assert out.ravel().tolist() == [float(x) for x in Xs] or np.allclose(out.ravel(), [float(x) for x in Xs], rtol=2e-16, atol=0)
