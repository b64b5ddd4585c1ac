"""Pins for the Scheme I 4M complex oracle (-m "not gpu"): the embedding
identity against numpy's complex product on small integers (exact), and the __float128 complex brute force
inside the Scheme I truncation bound of the embedded real problem."""
import numpy as np

import emugemm_inputs as G
from oracle import oracle as O
from test_oracle_oz1 import oz1_error_bound


def test_small_gaussian_integers_exact():
    rng = np.random.default_rng(3)
    A = rng.integers(-31, 32, size=(12, 20)) + 1j * rng.integers(-31, 32, size=(12, 20))
    B = rng.integers(-31, 32, size=(20, 9)) + 1j * rng.integers(-31, 32, size=(20, 9))
    Cin = rng.integers(-5, 6, size=(12, 9)) + 1j * rng.integers(-5, 6, size=(12, 9))
    for p in (3, 8):
        assert np.array_equal(O.zgemm_oz1_4m(A, B, p), A @ B)
    assert np.array_equal(O.zgemm_oz1_4m(A, B, 4, alpha=2 - 1j, beta=1j, Cin=Cin), (2 - 1j) * (A @ B) + 1j * Cin)


def test_vs_float128_complex_bruteforce_within_bound():
    m, n, k, p = 48, 40, 96, 6
    A, B = G.complex_pair(m, n, k, 0.5, 3)
    C = O.zgemm_oz1_4m(A, B, p)
    exact, _ = O.bf128_zgemm(A, B)
    Ae = np.block([[A.real, -A.imag], [A.imag, A.real]])
    Be = np.vstack([B.real, B.imag])
    bound = oz1_error_bound(Ae, Be, p)  # bound of the embedded real Scheme I problem, rows i / m + i = Re / Im
    assert (np.abs(C.real - exact.real) < bound[:m] + np.spacing(np.abs(exact.real))).all()
    assert (np.abs(C.imag - exact.imag) < bound[m:] + np.spacing(np.abs(exact.imag))).all()
    # one slice fewer is visibly worse: the bound is not vacuous
    C5 = O.zgemm_oz1_4m(A, B, p - 1)
    assert np.median(np.abs(C5 - exact)) > 20 * np.median(np.abs(C - exact))


def test_rows_of_the_embedding_share_exponents():
    A, _ = G.complex_pair(9, 4, 33, 2.0, 11)
    Ae = np.block([[A.real, -A.imag], [A.imag, A.real]])
    e = O.row_exponents(np.ascontiguousarray(Ae))
    assert np.array_equal(e[:9], e[9:]) and np.array_equal(e[:9], O.row_exponents_z(A))


def test_cgemm_oracles_exact_on_gaussian_integers_and_close_to_truth():
    rng = np.random.default_rng(9)
    A = (rng.integers(-31, 32, size=(10, 24)) + 1j * rng.integers(-31, 32, size=(10, 24))).astype(np.complex64)
    B = (rng.integers(-31, 32, size=(24, 7)) + 1j * rng.integers(-31, 32, size=(24, 7))).astype(np.complex64)
    want = (A.astype(np.complex128) @ B.astype(np.complex128)).astype(np.complex64)
    assert np.array_equal(O.cgemm_oz1_4m(A, B, 3), want)
    assert np.array_equal(O.cgemm_oz2_3m(A, B, 9), want)
    Az, Bz = G.complex_pair(20, 16, 64, 0.5, 4)
    Ac, Bc = Az.astype(np.complex64), Bz.astype(np.complex64)
    exact, absZ = O.bf128_zgemm(Ac.astype(np.complex128), Bc.astype(np.complex128))
    for got in (O.cgemm_oz1_4m(Ac, Bc, 4), O.cgemm_oz2_3m(Ac, Bc, 11)):
        assert (np.abs(got.astype(np.complex128) - exact) <= 8 * 2.0 ** -23 * absZ).all()


def test_four_products_equal_the_real_embedding():
    """The oracle states 4M as four separate real slice products; the same value must come out of ONE real Scheme I
    product on the embedding A' = [[Re A, -Im A], [Im A, Re A]], B' = [[Re B], [Im B]] (the form the CUDA path uses),
    bit for bit: rows i and m + i of A' share the exponent of row i of A, the digits of -Im A are the negated digits."""
    try:
        for bits, p, seed in ((7, 3, 5), (7, 6, 6), (7, 8, 7), (8, 4, 8), (8, 7, 9), (O.DIGITS_SIGNMAG, 3, 5), (O.DIGITS_SIGNMAG, 8, 7)):
            O.set_slice_bits(bits)
            A, B = G.complex_pair(21, 17, 50, 1.0, seed)
            m = A.shape[0]
            Ae = np.ascontiguousarray(np.block([[A.real, -A.imag], [A.imag, A.real]]))
            Be = np.ascontiguousarray(np.vstack([B.real, B.imag]))
            T = O.dgemm_oz1(Ae, Be, p)
            got = O.zgemm_oz1_4m(A, B, p)
            assert np.array_equal(got.real, T[:m]) and np.array_equal(got.imag, T[m:]), (bits, p)
    finally:
        O.set_slice_bits(7)
