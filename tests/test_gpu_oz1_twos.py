"""-m gpu parity tests, Scheme I with the DEFAULT two's-complement 7-bit digits (R24; form 0 of
emugemm_set_slice_form) and the switch to the sign-magnitude form (R1): digits and INT32 accumulators bit-exact against the oracle's R24 mode, final FP64 / FP32 within 2 ulp of
(|A||B|)_ij, the k-chunk bound of the form, batched and operand-handle calls, one full-size point."""
import numpy as np
import pytest

import emugemm_inputs as G
from gpu_util import assert_within_ulps

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import torch
    from oracle import oracle as O
    import paper_2606_25453_b200 as E
    h = E.EmuGemm()
    h.set_slice_bits(7)
    h.set_slice_form(0)          # the defaults, spelled out
    O.set_slice_bits(7)
    yield torch, O, h, E
    O.set_slice_bits(7)
    h.close()


def dev(torch, x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


@pytest.mark.parametrize("p", [1, 2, 3, 5, 7, 8])
@pytest.mark.parametrize("shape", [(256, 256, 256), (130, 70, 333)])
def test_digits_bit_exact(env, p, shape):
    torch, O, h, E = env
    m, n, k = shape
    A, B = G.real_pair(m, n, k, 2.0, 5)
    A[0, 0] = 0.0
    A[1, 1] = -np.abs(A[1]).max() * 3            # a negative row maximum
    A[2, 2] = np.abs(A[2]).max() * 1.999
    A[3, :] = -np.abs(A[3, :])                   # an all-negative row
    A[4, 5] = -2.0 ** -70 * np.abs(A[4]).max()   # truncates to zero (toward zero, not to -1)
    B[:, 1] = -np.abs(B[:, 1])
    SA, eA = h.dbg_oz1_slices(dev(torch, A), False, p)
    SB, eB = h.dbg_oz1_slices(dev(torch, B), True, p)
    oA, oB = O.row_exponents(A), O.col_exponents(B)
    assert np.array_equal(eA.cpu().numpy(), oA) and np.array_equal(eB.cpu().numpy(), oB)
    SAh, SBh = SA.cpu().numpy(), SB.cpu().numpy()
    assert np.array_equal(SAh, O.oz1_slices_rows(A, oA, p))
    assert np.array_equal(SBh, O.oz1_slices_cols(B, oB, p))
    if p > 1:
        assert SAh[1:].min() >= 0 and SBh[1:].min() >= 0   # every slice but the leading one is sign-free


def test_digits_f32_bit_exact(env):
    torch, O, h, E = env
    A, B = G.real_pair(100, 60, 200, 1.0, 4, dtype=np.float32)
    SA, _ = h.dbg_oz1_slices(dev(torch, A), False, 4)
    SB, _ = h.dbg_oz1_slices(dev(torch, B), True, 4)
    A64, B64 = A.astype(np.float64), B.astype(np.float64)
    assert np.array_equal(SA.cpu().numpy(), O.oz1_slices_rows(A64, O.row_exponents(A64), 4))
    assert np.array_equal(SB.cpu().numpy(), O.oz1_slices_cols(B64, O.col_exponents(B64), 4))


@pytest.mark.parametrize("p", [1, 2, 3, 4, 5, 6, 7, 8])
def test_int32_accumulators_bit_exact(env, p):
    torch, O, h, E = env
    m, n, k = (256, 320, 384) if p % 2 else (200, 150, 300)
    A, B = G.real_pair(m, n, k, 0.5, 100 + p)
    acc = h.dbg_oz1_accumulators(dev(torch, A), dev(torch, B), p).cpu().numpy()
    eA, eB = O.row_exponents(A), O.col_exponents(B)
    CS = O.oz1_accumulators(O.oz1_slices_rows(A, eA, p), O.oz1_slices_cols(B, eB, p))
    assert acc.shape == (1, p, m, n)
    assert np.array_equal(acc[0].astype(np.int64), CS)


@pytest.mark.parametrize("p,shape,phi", [(2, (256, 512, 256), 0.5), (3, (384, 320, 512), 0.5), (4, (129, 257, 130), 2.0),
                                         (5, (300, 200, 333), 2.0), (6, (300, 200, 333), 2.0), (7, (515, 130, 700), 2.0),
                                         (8, (128, 64, 128), 1.0), (8, (520, 300, 1000), 0.5)])
def test_dgemm_full_matrix(env, p, shape, phi):
    torch, O, h, E = env
    m, n, k = shape
    A, B = G.real_pair(m, n, k, phi, 1)
    C = torch.full((m, n), float("nan"), dtype=torch.float64, device="cuda")
    h.dgemm_oz1(dev(torch, A), dev(torch, B), C, p)
    _, absAB = O.bf128_dgemm(A, B)
    assert_within_ulps(C.cpu().numpy(), O.dgemm_oz1(A, B, p), absAB, 2, what=f"twos p={p} {shape}")


def test_alpha_beta_transposed_and_sgemm(env):
    torch, O, h, E = env
    m, n, k, p = 200, 136, 260, 7
    A, B, Cin = G.real_pair(m, n, k, 1.0, 9, with_c=True)
    Cd = dev(torch, Cin)
    h.dgemm_oz1(dev(torch, np.ascontiguousarray(A.T)), dev(torch, np.ascontiguousarray(B.T)), Cd, p, alpha=-1.5, beta=0.75,
                transa=True, transb=True)
    _, absAB = O.bf128_dgemm(A, B)
    assert_within_ulps(Cd.cpu().numpy(), O.dgemm_oz1(A, B, p, alpha=-1.5, beta=0.75, Cin=Cin), 1.5 * absAB + 0.75 * np.abs(Cin), 2)
    A32, B32 = G.real_pair(260, 200, 300, 1.0, 4, dtype=np.float32)
    C32 = torch.zeros((260, 200), dtype=torch.float32, device="cuda")
    h.sgemm_oz1(dev(torch, A32), dev(torch, B32), C32, 3)
    _, ab32 = O.bf128_dgemm(A32.astype(np.float64), B32.astype(np.float64))
    assert_within_ulps(C32.cpu().numpy(), O.sgemm_oz1(A32, B32, 3), ab32, 2, bits=23, what="sgemm twos p=3")


def test_chunk_bound_and_k_chunked(env):
    """R24: the leading digit reaches -128, so the fullest accumulator sums 2 pairs <= 128 * 127 and p - 2 pairs <= 127^2 per
    k: p = 8 gives 16,512 columns (R1: 16,640); k = 17,000 takes 2 chunks + the exact reduction.  Worst-case operands (every
    element the most negative value of its row / column) must not overflow INT32 at the bound."""
    torch, O, h, E = env
    for p in range(1, 9):
        per_k = 128 * 128 if p == 1 else 2 * 128 * 127 + (p - 2) * 127 * 127
        ck = E.oz1_chunk_k(p)
        assert ck % 128 == 0 and ck * per_k <= 2 ** 31 - 1 < (ck + 128) * per_k
    assert E.oz1_chunk_k(8) == 16512 and E.oz1_chunk_k(8, E.DIGITS_SIGN_MAGNITUDE) == 16640
    m, n, k, p = 64, 48, 17000, 8
    A, B = G.real_pair(m, n, k, 1.0, 4)
    C = torch.zeros((m, n), dtype=torch.float64, device="cuda")
    h.dgemm_oz1(dev(torch, A), dev(torch, B), C, p)
    assert_within_ulps(C.cpu().numpy(), O.dgemm_oz1(A, B, p), np.abs(A) @ np.abs(B), 2, what="twos chunked")
    # the extreme case of the bound: x = -(1 - 2^-52) 2^e everywhere -> leading digits -128, all lower digits 127... in BOTH operands
    k2 = 16512
    A2 = np.full((128, k2), -(1.0 - 2.0 ** -52))
    B2 = np.full((k2, 64), -(1.0 - 2.0 ** -52))
    acc = h.dbg_oz1_accumulators(dev(torch, A2), dev(torch, B2), 8).cpu().numpy()
    CS = O.oz1_accumulators(O.oz1_slices_rows(A2, O.row_exponents(A2), 8), O.oz1_slices_cols(B2, O.col_exponents(B2), 8))
    assert np.abs(CS).max() < 2 ** 31 and np.array_equal(acc[0].astype(np.int64), CS)


def test_batched_and_operand_handles(env):
    torch, O, h, E = env
    batch, m, n, k, p = 3, 129, 66, 300, 8
    rng = np.random.default_rng(17)
    A = (rng.random((batch, m, k)) - 0.5) * np.exp(rng.standard_normal((batch, m, k)))
    B = (rng.random((batch, k, n)) - 0.5) * np.exp(rng.standard_normal((batch, k, n)))
    C = torch.full((batch, m, n), float("nan"), dtype=torch.float64, device="cuda")
    h.dgemm_oz1_strided_batched(dev(torch, A), dev(torch, B), C, p)
    for b in range(batch):
        assert_within_ulps(C[b].cpu().numpy(), O.dgemm_oz1(A[b], B[b], p), np.abs(A[b]) @ np.abs(B[b]), 2, what=f"twos batched {b}")
    opA = h.decompose(E.OZ1, 0, dev(torch, A[0]), p)
    opB = h.decompose(E.OZ1, 1, dev(torch, B[0]), p)
    C2 = torch.empty((m, n), dtype=torch.float64, device="cuda")
    h.gemm_pre(opA, opB, C2)
    assert torch.equal(C2, C[0])
    # an operand decomposed in the other digit form must be refused, not silently mixed
    h0 = E.EmuGemm()
    h0.set_slice_form(1)
    try:
        opB0 = h0.decompose(E.OZ1, 1, dev(torch, B[0]), p)
        with pytest.raises(E.EmuGemmError):
            h.gemm_pre(opA, opB0, C2)
    finally:
        h0.close()


def test_form_switching_sign_magnitude_and_4m(env):
    """Form 1 = sign-magnitude digits (R1): bit-exact digits and 2-ulp parity against the oracle's R1 mode on the same handle type;
    8-bit digits have no forms; the 4M complex call runs in both 7-bit forms."""
    torch, O, h, E = env
    h2 = E.EmuGemm()
    try:
        h2.set_slice_bits(8)
        with pytest.raises(E.EmuGemmError):
            h2.set_slice_form(1)            # the forms exist for 7-bit digits only
        h2.set_slice_bits(7)
        h2.set_slice_form(1)
        O.set_slice_bits(O.DIGITS_SIGNMAG)
        A, B = G.real_pair(130, 70, 333, 2.0, 5)
        A[1, :] = -np.abs(A[1, :])
        SA, eA = h2.dbg_oz1_slices(dev(torch, A), False, 6)
        SAh = SA.cpu().numpy()
        assert np.array_equal(SAh, O.oz1_slices_rows(A, O.row_exponents(A), 6)) and SAh.min() >= -127 and SAh[1:].min() < 0
        C = torch.empty((130, 70), dtype=torch.float64, device="cuda")
        h2.dgemm_oz1(dev(torch, A), dev(torch, B), C, 6)
        assert_within_ulps(C.cpu().numpy(), O.dgemm_oz1(A, B, 6), np.abs(A) @ np.abs(B), 2, what="sign-magnitude form")
        # batched and operand-handle calls in the sign-magnitude form
        rng = np.random.default_rng(23)
        Ab = (rng.random((3, 100, 260)) - 0.5) * np.exp(rng.standard_normal((3, 100, 260)))
        Bb = (rng.random((3, 260, 70)) - 0.5) * np.exp(rng.standard_normal((3, 260, 70)))
        Cb = torch.full((3, 100, 70), float("nan"), dtype=torch.float64, device="cuda")
        h2.dgemm_oz1_strided_batched(dev(torch, Ab), dev(torch, Bb), Cb, 7)
        for b in range(3):
            assert_within_ulps(Cb[b].cpu().numpy(), O.dgemm_oz1(Ab[b], Bb[b], 7), np.abs(Ab[b]) @ np.abs(Bb[b]), 2, what=f"R1 batched {b}")
        opA, opB = h2.decompose(E.OZ1, 0, dev(torch, Ab[1]), 7), h2.decompose(E.OZ1, 1, dev(torch, Bb[1]), 7)
        Cp = torch.empty((100, 70), dtype=torch.float64, device="cuda")
        h2.gemm_pre(opA, opB, Cp)
        assert torch.equal(Cp, Cb[1])
        Az, Bz = G.complex_pair(40, 24, 100, 1.0, 3)
        absZ = (np.abs(Az.real) + np.abs(Az.imag)) @ (np.abs(Bz.real) + np.abs(Bz.imag))
        for form, code in ((1, O.DIGITS_SIGNMAG), (0, 7)):
            h2.set_slice_form(form)
            O.set_slice_bits(code)
            Cz = torch.zeros((40, 24), dtype=torch.complex128, device="cuda")
            h2.zgemm_oz1_4m(dev(torch, Az), dev(torch, Bz), Cz, 4)
            want = O.zgemm_oz1_4m(Az, Bz, 4)
            assert_within_ulps(Cz.cpu().numpy().real, want.real, absZ, 2, what=f"4M re form {form}")
            assert_within_ulps(Cz.cpu().numpy().imag, want.imag, absZ, 2, what=f"4M im form {form}")
    finally:
        O.set_slice_bits(7)
        h2.close()


def test_full_size_8192_p8_and_p4(env):
    torch, O, h, E = env
    size = 8192
    A, B = G.real_pair(size, size, size, 0.5, 1)
    dA, dB = dev(torch, A), dev(torch, B)
    rows, cols = G.sample_indices(size, 36, 7)[:48], G.sample_indices(size, 36, 8)[:48]
    for p in (8, 4):
        C = torch.full((size, size), float("nan"), dtype=torch.float64, device="cuda")
        h.dgemm_oz1(dA, dB, C, p)
        got = C[torch.from_numpy(rows).cuda()][:, torch.from_numpy(cols).cuda()].cpu().numpy()
        want = O.oz1_sampled(A, B, p, rows, cols)
        scale = np.abs(A[rows, :]) @ np.abs(B[:, cols])
        assert_within_ulps(got, want, scale, 2, what=f"twos 8192 p={p}")
        assert torch.isfinite(C).all()
